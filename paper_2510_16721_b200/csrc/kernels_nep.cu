// kernels_nep.cu -- K2, pass 1, for the NEP-shaped potential CFNEB_POT_NEP (include/cfneb.h): the descriptor network of
// kernels_dn.cu widened to the shape and cost of the paper's force field proper ("NEP-trained force field";
// its evaluation is the 10^6 atom-steps per second the paper quotes): separate radial and angular cut-offs,
// two atom types with type-pair expansion coefficients, basis sizes and descriptor counts as parameters, Legendre
// orders up to 4, one network of up to 64 neurons per type.  Seeded weights (the trained ones are not available):
// cost and data flow, no physics.  It enters the path through the partial forces p^ij = dU_i/dr^ij of Eq. 5; pass 2
// (f^ij = p^ij - p^ji, F_i, virial of Eq. 8) is the kernel the other many-body potentials use (kernels_sw.cu).
//   f_k(r; rc) = 1/2 [T_k(x) + 1] fc(r; rc),  x = 2 (r/rc - 1)^2 - 1,  fc = 1/2 [1 + cos(pi r/rc)]
//   g^R_n = sum_k cR[I][J][n][k] f_k(r; rc_r),   g^A_n = sum_k cA[I][J][n][k] f_k(r; rc_a)      (I, J: types of i, j)
//   q_n    = sum_j g^R_n(r_ij)                                                                  n < n_r
//   q_{nl} = sum_j sum_k g^A_n(r_ij) g^A_n(r_ik) P_l(cos theta_jik)                             n < n_a, l = 1..L
//   U_i    = sum_mu W1[I][mu] tanh(sum_d W0[I][mu][d] q_d - b0[I][mu])
// As in kernels_dn.cu the double sum over the environment is never formed: with u = r/|r| and the moments
//   S^(l)_n = sum_j g^A_n(r_ij) u_ij^(x)l     (l = 0..4: 1 + 3 + 6 + 10 + 15 = 35 independent components per n)
// A_l = sum_jk g g (u_j.u_k)^l = |S^(l)|^2 and q_{n1} = A_1, q_{n2} = 3/2 A_2 - 1/2 A_0, q_{n3} = 5/2 A_3 - 3/2 A_1,
// q_{n4} = (35 A_4 - 30 A_2 + 3 A_0)/8.
//
// Work split (round 1's descriptor kernel held all channels of an atom in one thread: 236 registers, 8 warps per
// multiprocessor).  FOUR LANES PER ATOM: lane q of a quad owns the angular channels n = q, q + 4 and the radial
// descriptors n = q, q + 4, and a quarter of the neurons.  All four walk the same list rows (their loads coalesce into
// one request); each accumulates the 35 moments of ONE channel per walk in registers, parks them in a scratch array
// (one 280-byte column per atom and channel), the quad exchanges descriptors and descriptor gradients by shuffles, and
// a second walk per channel evaluates phi_n(u) = sum_c G_nc u^c and its gradient and sums the four lanes' partial
// forces by two shuffle steps before one lane writes them.  Network weights and expansion coefficients sit in shared
// memory.  No per-thread environment array, hence no limit on the atoms inside the cut-offs but the list capacity.
#include "cfneb_internal.cuh"
#include "nep_poly.cuh"
#include "trig01.cuh"

namespace cfn {

constexpr int kNepMaxN = 8, kNepMaxK = 12, kNepMaxH = 64, kNepMaxL = 4;
constexpr int kNepThreads = 128;  // 32 atoms x 4 lanes

struct NepShape {
    int nr, na, kr, ka, L, H, T, D;
};
__host__ __device__ inline NepShape nep_shape(const double *pot) {
    NepShape s;
    s.nr = (int)pot[2]; s.na = (int)pot[3]; s.kr = (int)pot[4]; s.ka = (int)pot[5];
    s.L = (int)pot[6]; s.H = (int)pot[7]; s.T = (int)pot[8];
    s.D = s.nr + s.na * s.L;
    return s;
}
// layout of Dev::dn_w for this potential: per type [W0 H*D | b0 H | W1 H], then cR [T][T][nr][kr], then cA [T][T][na][ka]
__host__ __device__ inline int nep_net_size(const NepShape &s) { return s.H * s.D + 2 * s.H; }
__host__ __device__ inline int nep_weights_size(const NepShape &s) {
    return s.T * nep_net_size(s) + s.T * s.T * (s.nr * s.kr + s.na * s.ka);
}

// Chebyshev radial basis f_k and df_k/dr for k < K (recurrence); t = r / rc in (0, 1)
template <int KMAX>
__device__ __forceinline__ void nep_basis(double t, double irc, int K, double (&f)[KMAX], double (&df)[KMAX]) {
    double sn, cs;
    sincospi01(t, sn, cs);
    const double fc = 0.5 + 0.5 * cs, dfc = -0.5 * sn * (3.14159265358979323846 * irc);
    const double x = 2.0 * (t - 1.0) * (t - 1.0) - 1.0, dx_dr = 4.0 * (t - 1.0) * irc;
    double Tm = 1.0, Tk = x, dTm = 0.0, dTk = 1.0;  // T_{k-1}, T_k and derivatives with respect to x (k = 1)
#pragma unroll
    for (int k = 0; k < KMAX; ++k) {
        if (k < K) {
            const double Tv = k == 0 ? 1.0 : Tk, dTv = k == 0 ? 0.0 : dTk;
            const double g = 0.5 * (Tv + 1.0);
            f[k] = g * fc;
            df[k] = 0.5 * dTv * dx_dr * fc + g * dfc;
            if (k >= 1) {
                const double Tn = 2.0 * x * Tk - Tm, dTn = 2.0 * Tk + 2.0 * x * dTk - dTm;
                Tm = Tk; Tk = Tn; dTm = dTk; dTk = dTn;
            }
        } else {
            f[k] = 0.0;
            df[k] = 0.0;
        }
    }
}

__global__ void __launch_bounds__(kNepThreads, 3) nep_partial_kernel(Dev d, int p_lo) {
    int p;
    if (!image_of(blockIdx.y, p_lo, d.ctl->P, p)) return;
    const int slot = d.order[p];
    extern __shared__ double sW[];  // all weights of the potential
    __shared__ double sh[9];
    __shared__ double red[64];
    const NepShape sp = nep_shape(d.pot);
    const int nW = nep_weights_size(sp);
    if (threadIdx.x < 9) sh[threadIdx.x] = d.geom[slot].h[threadIdx.x];
    for (int t = threadIdx.x; t < nW; t += blockDim.x) sW[t] = d.dn_w[t];
    __syncthreads();
    const int q = threadIdx.x & 3;                                     // lane of the quad
    const int i = blockIdx.x * (kNepThreads / 4) + (threadIdx.x >> 2);  // atom of the quad
    const bool valid = i < d.N;
    const int ic = valid ? i : 0;
    const unsigned quad_mask = 0xFu << ((threadIdx.x & 31) & ~3);  // the quad's lanes: its shuffles run inside loops whose
                                                                   // trip count (the atom's list length) differs between quads
    const double rcr = d.pot[0], rca = d.pot[1], rcr2 = rcr * rcr, rca2 = rca * rca, ircr = 1.0 / rcr, irca = 1.0 / rca;
    const int I = d.types[ic];
    const double *net = sW + I * nep_net_size(sp);
    const double *W0 = net, *b0 = net + sp.H * sp.D, *W1 = b0 + sp.H;
    const double *cRb = sW + sp.T * nep_net_size(sp) + (size_t)I * sp.T * sp.nr * sp.kr;   // [J][n][k]
    const double *cAb = sW + sp.T * nep_net_size(sp) + sp.T * sp.T * sp.nr * sp.kr + (size_t)I * sp.T * sp.na * sp.ka;
    const double4 *Rc = d.Rc + (size_t)slot * d.Npad;
    const uint32_t *lp = d.nbr_list + (size_t)slot * d.cap * d.Npad + ic;
    double *part = d.part + (size_t)slot * d.cap * 3 * d.Npad + ic;  // part[(k * 3 + m) * Npad]
    double *scr = d.nep_S + ((size_t)slot * sp.na * kNepC) * d.Npad + ic;  // scr[(n * kNepC + c) * Npad]
    const double4 ri = Rc[ic];
    const int cnt = valid ? live_rows(d, slot, ic) : 0;  // rows past it cannot be in range

    auto pair_vec = [&](int k, int &J, double &dx, double &dy, double &dz) {
        const uint32_t e = lp[(size_t)k * d.Npad];
        const uint32_t j = e & kIdxMask, code = e >> kShiftBits;
        const double4 rj = Rc[j];
        J = d.types[j];
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

    // ---- walk 1 (one per angular channel of this lane; the first also takes the radial descriptors) ----
    double qR[2] = {0.0, 0.0};               // radial descriptors n = q, q + 4
    double qA[2][kNepMaxL] = {};             // angular descriptors of the channels n = q, q + 4
    const int npass = (sp.na + 3) / 4;
    for (int pass = 0; pass < npass; ++pass) {
        const int n = q + 4 * pass;
        const bool own = n < sp.na;
        double S[kNepC];
#pragma unroll
        for (int c = 0; c < kNepC; ++c) S[c] = 0.0;
        for (int k = 0; k < cnt; ++k) {
            int J;
            double dx, dy, dz;
            const double r2 = pair_vec(k, J, dx, dy, dz);
            if (!(r2 < rcr2)) continue;
            const double inv = rsqrt(r2), r = r2 * inv;
            if (pass == 0) {
                double f[kNepMaxK], df[kNepMaxK];
                nep_basis<kNepMaxK>(r * ircr, ircr, sp.kr, f, df);
#pragma unroll
                for (int h2 = 0; h2 < 2; ++h2) {
                    const int nn = q + 4 * h2;
                    if (nn < sp.nr) {
                        const double *c = cRb + ((size_t)J * sp.nr + nn) * sp.kr;
                        double g = 0.0;
                        for (int b = 0; b < sp.kr; ++b) g += c[b] * f[b];
                        qR[h2] += g;
                    }
                }
            }
            if (own && r2 < rca2) {
                double f[kNepMaxK], df[kNepMaxK], m[kNepC];
                nep_basis<kNepMaxK>(r * irca, irca, sp.ka, f, df);
                const double *c = cAb + ((size_t)J * sp.na + n) * sp.ka;
                double g = 0.0;
                for (int b = 0; b < sp.ka; ++b) g += c[b] * f[b];
                nep_monomials(dx * inv, dy * inv, dz * inv, m);
#pragma unroll
                for (int cc = 0; cc < kNepC; ++cc) S[cc] += g * m[cc];
            }
        }
        if (own && valid) {
            double A[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
            for (int cc = 0; cc < kNepC; ++cc) {
                const int l = cc < 1 ? 0 : cc < 4 ? 1 : cc < 10 ? 2 : cc < 20 ? 3 : 4;
                A[l] += kNepMult[cc] * S[cc] * S[cc];
                scr[(size_t)(n * kNepC + cc) * d.Npad] = S[cc];
            }
            qA[pass][0] = A[1];
            qA[pass][1] = 1.5 * A[2] - 0.5 * A[0];
            qA[pass][2] = 2.5 * A[3] - 1.5 * A[1];
            qA[pass][3] = 0.125 * (35.0 * A[4] - 30.0 * A[2] + 3.0 * A[0]);
        }
    }

    // ---- the network: every lane needs all descriptors; each takes the neurons mu = q, q + 4, ... ----
    // descriptor d lives in lane (d mod 4 for radial n = d; angular channel n -> lane n mod 4): gather by quad shuffles
    double ui = 0.0;
    double FdR[2] = {0.0, 0.0}, FdA[2][kNepMaxL] = {};
    {
        double z[kNepMaxH / 4];
#pragma unroll
        for (int t = 0; t < kNepMaxH / 4; ++t) {
            const int mu = q + 4 * t;
            z[t] = mu < sp.H ? -b0[mu] : 0.0;
        }
        const int base_lane = (threadIdx.x & 31) & ~3;
        for (int dsc = 0; dsc < sp.D; ++dsc) {
            // owner lane and register of descriptor dsc
            int ol, hh, ll = 0;
            bool radial = dsc < sp.nr;
            if (radial) { ol = dsc & 3; hh = dsc >> 2; }
            else { const int n = (dsc - sp.nr) / sp.L; ll = (dsc - sp.nr) % sp.L; ol = n & 3; hh = n >> 2; }
            double mine = radial ? (hh ? qR[1] : qR[0]) : (hh ? qA[1][0] : qA[0][0]);
            if (!radial) {
                if (ll == 1) mine = hh ? qA[1][1] : qA[0][1];
                if (ll == 2) mine = hh ? qA[1][2] : qA[0][2];
                if (ll == 3) mine = hh ? qA[1][3] : qA[0][3];
            }
            const double v = __shfl_sync(quad_mask, mine, base_lane + ol);
#pragma unroll
            for (int t = 0; t < kNepMaxH / 4; ++t) {
                const int mu = q + 4 * t;
                if (mu < sp.H) z[t] += W0[mu * sp.D + dsc] * v;
            }
        }
        double gmu[kNepMaxH / 4];
#pragma unroll
        for (int t = 0; t < kNepMaxH / 4; ++t) {
            const int mu = q + 4 * t;
            gmu[t] = 0.0;
            if (mu < sp.H) {
                const double th = tanh(z[t]);
                ui += W1[mu] * th;
                gmu[t] = W1[mu] * (1.0 - th * th);
            }
        }
        // dU/dq_d = sum_mu gmu W0[mu][d]: partial over this lane's neurons, summed over the quad, kept by the owner
        for (int dsc = 0; dsc < sp.D; ++dsc) {
            double v = 0.0;
#pragma unroll
            for (int t = 0; t < kNepMaxH / 4; ++t) {
                const int mu = q + 4 * t;
                if (mu < sp.H) v += gmu[t] * W0[mu * sp.D + dsc];
            }
            v += __shfl_xor_sync(quad_mask, v, 1);
            v += __shfl_xor_sync(quad_mask, v, 2);
            if (dsc < sp.nr) {
                if ((dsc & 3) == q) { if (dsc >> 2) FdR[1] = v; else FdR[0] = v; }
            } else {
                const int n = (dsc - sp.nr) / sp.L, ll = (dsc - sp.nr) % sp.L;
                if ((n & 3) == q) {
#pragma unroll
                    for (int l2 = 0; l2 < kNepMaxL; ++l2)
                        if (l2 == ll) { if (n >> 2) FdA[1][l2] = v; else FdA[0][l2] = v; }
                }
            }
        }
        ui += __shfl_xor_sync(quad_mask, ui, 1);
        ui += __shfl_xor_sync(quad_mask, ui, 2);
        if (q != 0 || !valid) ui = 0.0;  // one lane per atom carries the site energy
    }

    // ---- walk 2 (one per pass): partial forces.  Lane sums of the quad are combined per list row ----
    for (int pass = 0; pass < npass; ++pass) {
        const int n = q + 4 * pass;
        const bool own = n < sp.na;
        double G[kNepC];  // dU/dS_nc = 2 coef_l mult_c S_nc
        {
            const double *F = pass ? FdA[1] : FdA[0];
            const double F1 = F[0], F2 = sp.L > 1 ? F[1] : 0.0, F3 = sp.L > 2 ? F[2] : 0.0, F4 = sp.L > 3 ? F[3] : 0.0;
            const double cf[5] = {-0.5 * F2 + 0.375 * F4, F1 - 1.5 * F3, 1.5 * F2 - 3.75 * F4, 2.5 * F3, 4.375 * F4};
#pragma unroll
            for (int cc = 0; cc < kNepC; ++cc) {
                const int l = cc < 1 ? 0 : cc < 4 ? 1 : cc < 10 ? 2 : cc < 20 ? 3 : 4;
                G[cc] = (own && valid) ? 2.0 * cf[l] * kNepMult[cc] * scr[(size_t)(n * kNepC + cc) * d.Npad] : 0.0;
            }
        }
        for (int k = 0; k < cnt; ++k) {
            int J;
            double dx, dy, dz;
            const double r2 = pair_vec(k, J, dx, dy, dz);
            double px = 0.0, py = 0.0, pz = 0.0;
            if (r2 < rcr2) {
                const double inv = rsqrt(r2), r = r2 * inv;
                const double x = dx * inv, y = dy * inv, z = dz * inv;
                if (pass == 0) {  // radial descriptors: sum_n Fd_n g'_n(r) u
                    double f[kNepMaxK], df[kNepMaxK];
                    nep_basis<kNepMaxK>(r * ircr, ircr, sp.kr, f, df);
                    double s = 0.0;
#pragma unroll
                    for (int h2 = 0; h2 < 2; ++h2) {
                        const int nn = q + 4 * h2;
                        if (nn < sp.nr) {
                            const double *c = cRb + ((size_t)J * sp.nr + nn) * sp.kr;
                            double dg = 0.0;
                            for (int b = 0; b < sp.kr; ++b) dg += c[b] * df[b];
                            s += (h2 ? FdR[1] : FdR[0]) * dg;
                        }
                    }
                    px = s * x; py = s * y; pz = s * z;
                }
                if (own && r2 < rca2) {
                    double f[kNepMaxK], df[kNepMaxK], m[kNepC];
                    nep_basis<kNepMaxK>(r * irca, irca, sp.ka, f, df);
                    const double *c = cAb + ((size_t)J * sp.na + n) * sp.ka;
                    double g = 0.0, dg = 0.0;
                    for (int b = 0; b < sp.ka; ++b) { g += c[b] * f[b]; dg += c[b] * df[b]; }
                    nep_monomials(x, y, z, m);  // only the monomials of degree <= 3 are read below
                    double gl[4][3];
                    nep_poly_grad(G, m, gl);
                    double phi = G[0], ug = 0.0, gx = 0.0, gy = 0.0, gz = 0.0;
#pragma unroll
                    for (int l = 0; l < 4; ++l) {  // u . grad phi_l = l phi_l (Euler)
                        const double t = x * gl[l][0] + y * gl[l][1] + z * gl[l][2];
                        ug += t;
                        phi += t * (1.0 / (l + 1));
                        gx += gl[l][0]; gy += gl[l][1]; gz += gl[l][2];
                    }
                    const double gi = g * inv, dphi = dg * phi;
                    px += dphi * x + gi * (gx - ug * x);
                    py += dphi * y + gi * (gy - ug * y);
                    pz += dphi * z + gi * (gz - ug * z);
                }
            }
            // the quad's four contributions; lane m < 3 then owns component m
            px += __shfl_xor_sync(quad_mask, px, 1); px += __shfl_xor_sync(quad_mask, px, 2);
            py += __shfl_xor_sync(quad_mask, py, 1); py += __shfl_xor_sync(quad_mask, py, 2);
            pz += __shfl_xor_sync(quad_mask, pz, 1); pz += __shfl_xor_sync(quad_mask, pz, 2);
            if (q < 3) {
                double *o = part + (size_t)(k * 3 + q) * d.Npad;
                const double v = q == 0 ? px : q == 1 ? py : pz;
                *o = pass ? *o + v : v;
            }
        }
    }
    double ui_lo = 0.0;
    block_sum_dd(ui, ui_lo, red);
    if (threadIdx.x == 0) {
        double *out = d.part_force + ((size_t)slot * d.nblk_force + blockIdx.x) * kNForcePart;
        out[7] = ui;
        out[9] = ui_lo;
    }
}

int nep_weight_count(const double *pot) { return nep_weights_size(nep_shape(pot)); }

// The weight stream of include/cfneb.h (SplitMix64 from the seed), in the layout of Dev::dn_w.  Host.
void nep_fill_weights(const double *pot, double *w) {
    const NepShape s = nep_shape(pot);
    uint64_t state = (uint64_t)pot[9];
    auto next = [&]() {
        uint64_t z = (state += 0x9E3779B97F4A7C15ull);
        z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
        z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
        z ^= z >> 31;
        return 2.0 * ((double)(z >> 11) * (1.0 / 9007199254740992.0)) - 1.0;
    };
    for (int I = 0; I < s.T; ++I) {
        double *net = w + (size_t)I * nep_net_size(s);
        for (int t = 0; t < s.H * s.D; ++t) net[t] = next() * ((t % s.D) < s.nr ? 0.04 : 0.004);
        for (int t = 0; t < s.H; ++t) net[s.H * s.D + t] = 0.5 * next();
        for (int t = 0; t < s.H; ++t) net[s.H * s.D + s.H + t] = next();
    }
    double *c = w + (size_t)s.T * nep_net_size(s);
    const int nc = s.T * s.T * (s.nr * s.kr + s.na * s.ka);
    for (int t = 0; t < nc; ++t) c[t] = next();
}

void launch_force_nep(const Dev &d, int p_lo, cudaStream_t st) {
    const int nimg = images_in_grid(d.S, p_lo);
    if (nimg <= 0) return;
    dim3 grid(d.nblk_force, nimg);
    const size_t smem = (size_t)nep_weight_count(d.pot) * sizeof(double);
    static bool attr_set = false;
    if (!attr_set) {
        cudaFuncSetAttribute(nep_partial_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
        attr_set = true;
    }
    nep_partial_kernel<<<grid, kNepThreads, smem, st>>>(d, p_lo);
    launch_pair_forces_manybody(d, p_lo, st);
}

}  // namespace cfn

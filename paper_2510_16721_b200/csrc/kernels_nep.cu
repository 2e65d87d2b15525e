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
// a quarter of the neurons.  The list is walked four rows at a time, ONE ROW PER LANE: a lane forms the pair vector, the
// two radial bases and the expansions g_n of its row once, then the rows go round the quad by shuffles and every lane
// adds each row to the 35 moments of its own channel (registers); the moments are parked in a scratch array (one
// 280-byte column per atom and channel), the quad exchanges descriptors and descriptor gradients by shuffles, and a
// second walk of the same shape evaluates phi_n(u) = sum_c G_nc u^c and its gradient per channel and hands the three
// components back to the row's lane, which writes them once.  Network weights and expansion coefficients sit in shared
// memory.  No per-thread environment array, hence no limit on the atoms inside the cut-offs but the list capacity.
#include "cfneb_internal.cuh"
#include "nep_poly.cuh"
#include "trig01.cuh"

namespace cfn {

constexpr int kNepMaxN = 8, kNepMaxK = 12, kNepMaxH = 64, kNepMaxL = 4;
constexpr int kNepThreads = 128;  // 32 atoms x 4 lanes
#ifndef CFNEB_NEP_BLOCKS
#define CFNEB_NEP_BLOCKS 2
#endif

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

// KMAX: basis functions held per row (the smallest of 4, 8, 12 that covers k_r and k_a): the loops over them are
// unrolled so that the basis stays in registers.
template <int KMAX>
__global__ void __launch_bounds__(kNepThreads, CFNEB_NEP_BLOCKS) nep_partial_kernel(Dev d, int p_lo) {
    int p;
    if (!image_of(blockIdx.y, p_lo, d.ctl->P, p)) return;
    const int slot = d.order[p];
    extern __shared__ double sW[];  // all weights of the potential
    __shared__ double sh[9];
    __shared__ double red[64];
    const NepShape sp = nep_shape(d.pot);
    const int nNet = sp.T * nep_net_size(sp);
    if (threadIdx.x < 9) sh[threadIdx.x] = d.geom[slot].h[threadIdx.x];
    for (int t = threadIdx.x; t < nNet; t += blockDim.x) sW[t] = d.dn_w[t];
    // expansion coefficients zero-padded to [T][T][8][KMAX] (radial, then angular): the loops over channels and basis
    // functions then run to their compile-time bounds with no guards, and a row of coefficients is KMAX aligned doubles
    double *cRp = sW + ((nNet + 1) & ~1), *cAp = cRp + sp.T * sp.T * kNepMaxN * KMAX;
    for (int t = threadIdx.x; t < sp.T * sp.T * kNepMaxN * KMAX; t += blockDim.x) {
        const int b = t % KMAX, nn = (t / KMAX) % kNepMaxN, IJ = t / (KMAX * kNepMaxN);
        cRp[t] = (nn < sp.nr && b < sp.kr) ? d.dn_w[nNet + (IJ * sp.nr + nn) * sp.kr + b] : 0.0;
        cAp[t] = (nn < sp.na && b < sp.ka) ? d.dn_w[nNet + sp.T * sp.T * sp.nr * sp.kr + (IJ * sp.na + nn) * sp.ka + b] : 0.0;
    }
    __syncthreads();
    const int q = threadIdx.x & 3;                                     // lane of the quad
    const int i = blockIdx.x * (kNepThreads / 4) + (threadIdx.x >> 2);  // atom of the quad
    const bool valid = i < d.N;
    const int ic = valid ? i : 0;
    const unsigned quad_mask = 0xffffffffu;  // see cnt_w below
    const double rcr = d.pot[0], rca = d.pot[1], rcr2 = rcr * rcr, rca2 = rca * rca, ircr = 1.0 / rcr, irca = 1.0 / rca;
    const int I = d.types[ic];
    const double *net = sW + I * nep_net_size(sp);
    const double *W0 = net, *b0 = net + sp.H * sp.D, *W1 = b0 + sp.H;
    const double *cRb = cRp + (size_t)I * sp.T * kNepMaxN * KMAX;   // [J][n][k], padded
    const double *cAb = cAp + (size_t)I * sp.T * kNepMaxN * KMAX;
    const double4 *Rc = d.Rc + (size_t)slot * d.Npad;
    const uint32_t *lp = d.nbr_list + (size_t)slot * d.cap * d.Npad + ic;
    double *part = d.part + (size_t)slot * d.cap * 3 * d.Npad + ic;  // part[(k * 3 + m) * Npad]
    double *scr = d.nep_S + ((size_t)slot * sp.na * kNepC) * d.Npad + ic;  // scr[(n * kNepC + c) * Npad]
    const double4 ri = Rc[ic];
    const int cnt = valid ? live_rows(d, slot, ic) : 0;  // rows past it cannot be in range
    // every loop over list rows runs to the longest list of the warp (rows past a quad's own count are skipped by
    // `kk < cnt`): all 32 lanes reach every shuffle, so the shuffles take the full mask
    const int cnt_w = __reduce_max_sync(0xffffffffu, cnt);

    // The rows of a lane (kk = q, q + 4, ...) are software-pipelined: the list entry two rows ahead and the neighbour's
    // sector and type one row ahead are in flight while a row is evaluated (two resident warps per scheduler cannot
    // hide the two dependent loads otherwise).  Rows past the end stand in with the atom itself and are never used.
    uint32_t e_nn, e_n;
    double4 rj_n;
    int J_n;
    auto walk_begin = [&]() {
        e_n = q < cnt ? lp[(size_t)q * d.Npad] : (uint32_t)ic | (kCodeCenter << kShiftBits);
        e_nn = q + 4 < cnt ? lp[(size_t)(q + 4) * d.Npad] : e_n;
        rj_n = Rc[e_n & kIdxMask];
        J_n = d.types[e_n & kIdxMask];
    };
    auto pair_vec = [&](int k, int &J, double &dx, double &dy, double &dz) {  // row k of this lane; advances the pipeline
        const uint32_t code = e_n >> kShiftBits;
        const double4 rj = rj_n;
        J = J_n;
        e_n = e_nn;
        e_nn = k + 8 < cnt ? lp[(size_t)(k + 8) * d.Npad] : e_n;
        rj_n = Rc[e_n & kIdxMask];
        J_n = d.types[e_n & kIdxMask];
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

    const int base_lane = (threadIdx.x & 31) & ~3;
    auto sel4 = [](const double (&a)[4], int c) { return c == 0 ? a[0] : c == 1 ? a[1] : c == 2 ? a[2] : a[3]; };
    auto shf = [&](double v, int src) { return __shfl_sync(quad_mask, v, base_lane + src); };
    auto quad_sum = [&](double v) {
        v += __shfl_xor_sync(quad_mask, v, 1);
        return v + __shfl_xor_sync(quad_mask, v, 2);
    };

    // ---- walk 1: the list is taken four rows at a time, ONE ROW PER LANE: the lane forms the pair vector, the radial
    // basis and the expansions g_n of its row (nothing of that is done four times), then the rows go round the quad
    // (step t: lane q takes the row of lane q + t) and each lane adds every row to the moments of its own channel ----
    double qR[kNepMaxN];                      // radial descriptors: partial sums over this lane's rows, then all of them
#pragma unroll
    for (int n = 0; n < kNepMaxN; ++n) qR[n] = 0.0;
    double qA[2][kNepMaxL] = {};              // angular descriptors of the channels n = q, q + 4
    const int npass = (sp.na + 3) / 4;
    for (int pass = 0; pass < npass; ++pass) {
        const int n = q + 4 * pass;
        const bool own = n < sp.na;
        double S[kNepC];
#pragma unroll
        for (int c = 0; c < kNepC; ++c) S[c] = 0.0;
        walk_begin();
        for (int k0 = 0; k0 < cnt_w; k0 += 4) {
            const int kk = k0 + q;
            int J = 0;
            double dx = 0.0, dy = 0.0, dz = 0.0, r2 = 1e300;
            if (kk < cnt) r2 = pair_vec(kk, J, dx, dy, dz);
            double x = 0.0, y = 0.0, z = 0.0, g4[4] = {0.0, 0.0, 0.0, 0.0};
            if (r2 < rcr2) {
                const double inv = rsqrt(r2), r = r2 * inv;
                x = dx * inv; y = dy * inv; z = dz * inv;
                if (pass == 0) {
                    double f[KMAX], df[KMAX];
                    nep_basis<KMAX>(r * ircr, ircr, sp.kr, f, df);
                    const double *c = cRb + (size_t)J * kNepMaxN * KMAX;
#pragma unroll
                    for (int nn = 0; nn < kNepMaxN; ++nn) {
                        double g = 0.0;
#pragma unroll
                        for (int b = 0; b < KMAX; ++b) g += c[nn * KMAX + b] * f[b];
                        qR[nn] += g;
                    }
                }
                if (r2 < rca2) {
                    double f[KMAX], df[KMAX];
                    nep_basis<KMAX>(r * irca, irca, sp.ka, f, df);
#pragma unroll
                    for (int c4 = 0; c4 < 4; ++c4) {
                        const double *c = cAb + ((size_t)J * kNepMaxN + 4 * pass + c4) * KMAX;
                        double g = 0.0;
#pragma unroll
                        for (int b = 0; b < KMAX; ++b) g += c[b] * f[b];
                        g4[c4] = g;
                    }
                }
            }
            const double inA = r2 < rca2 ? 1.0 : 0.0;
#pragma unroll
            for (int t = 0; t < 4; ++t) {
                const int src = (q + t) & 3;
                // the value lane src wants from this lane in step t is the g of ITS channel: lane src = q + t reads q's
                // register, so q presents g4[(q - t) & 3]... seen from the reader: it reads g4[own channel] of lane src
                const double gs = t == 0 ? sel4(g4, q) : shf(sel4(g4, (q - t) & 3), src);
                const double xs = t == 0 ? x : shf(x, src), ys = t == 0 ? y : shf(y, src), zs = t == 0 ? z : shf(z, src);
                const double as = t == 0 ? inA : shf(inA, src);
                if (own && as != 0.0) {
                    double m[kNepC];
                    nep_monomials(xs, ys, zs, m);
#pragma unroll
                    for (int cc = 0; cc < kNepC; ++cc) S[cc] += gs * m[cc];
                }
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
#pragma unroll
    for (int n = 0; n < kNepMaxN; ++n) qR[n] = quad_sum(qR[n]);  // every lane now holds all radial descriptors

    // ---- the network: each lane takes the neurons mu = q, q + 4, ...; the angular descriptors come from their owners ----
    double ui = 0.0;
    double FdR[kNepMaxN], FdA[2][kNepMaxL] = {};
#pragma unroll
    for (int n = 0; n < kNepMaxN; ++n) FdR[n] = 0.0;
    {
        double zt[kNepMaxH / 4];
#pragma unroll
        for (int t = 0; t < kNepMaxH / 4; ++t) {
            const int mu = q + 4 * t;
            zt[t] = mu < sp.H ? -b0[mu] : 0.0;
        }
        for (int dsc = 0; dsc < sp.D; ++dsc) {
            double v;
            if (dsc < sp.nr) {
                v = 0.0;
#pragma unroll
                for (int n = 0; n < kNepMaxN; ++n)
                    if (n == dsc) v = qR[n];
            } else {
                const int n = (dsc - sp.nr) / sp.L, ll = (dsc - sp.nr) % sp.L, hh = n >> 2;
                double mine = hh ? qA[1][0] : qA[0][0];
                if (ll == 1) mine = hh ? qA[1][1] : qA[0][1];
                if (ll == 2) mine = hh ? qA[1][2] : qA[0][2];
                if (ll == 3) mine = hh ? qA[1][3] : qA[0][3];
                v = shf(mine, n & 3);
            }
#pragma unroll
            for (int t = 0; t < kNepMaxH / 4; ++t) {
                const int mu = q + 4 * t;
                if (mu < sp.H) zt[t] += W0[mu * sp.D + dsc] * v;
            }
        }
        double gmu[kNepMaxH / 4];
#pragma unroll
        for (int t = 0; t < kNepMaxH / 4; ++t) {
            const int mu = q + 4 * t;
            gmu[t] = 0.0;
            if (mu < sp.H) {
                const double th = tanh(zt[t]);
                ui += W1[mu] * th;
                gmu[t] = W1[mu] * (1.0 - th * th);
            }
        }
        // dU/dq_d = sum_mu gmu W0[mu][d]: partial over this lane's neurons, summed over the quad
        for (int dsc = 0; dsc < sp.D; ++dsc) {
            double v = 0.0;
#pragma unroll
            for (int t = 0; t < kNepMaxH / 4; ++t) {
                const int mu = q + 4 * t;
                if (mu < sp.H) v += gmu[t] * W0[mu * sp.D + dsc];
            }
            v = quad_sum(v);
            if (dsc < sp.nr) {
#pragma unroll
                for (int n = 0; n < kNepMaxN; ++n)
                    if (n == dsc) FdR[n] = v;  // all lanes keep the radial ones
            } else {
                const int n = (dsc - sp.nr) / sp.L, ll = (dsc - sp.nr) % sp.L;
                if ((n & 3) == q) {
#pragma unroll
                    for (int l2 = 0; l2 < kNepMaxL; ++l2)
                        if (l2 == ll) { if (n >> 2) FdA[1][l2] = v; else FdA[0][l2] = v; }
                }
            }
        }
        ui = quad_sum(ui);
        if (q != 0 || !valid) ui = 0.0;  // one lane per atom carries the site energy
    }

    // ---- walk 2 (one per pass), again one row per lane: the lane prepares its row (pair vector, bases, g_n and g_n'
    // of the pass's four channels, the radial part of the partial force), the rows go round the quad, every lane
    // evaluates ITS channel's polynomial for each row and hands the three components back to the row's lane ----
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
        walk_begin();
        for (int k0 = 0; k0 < cnt_w; k0 += 4) {
            const int kk = k0 + q;
            int J = 0;
            double dx = 0.0, dy = 0.0, dz = 0.0, r2 = 1e300;
            if (kk < cnt) r2 = pair_vec(kk, J, dx, dy, dz);
            double x = 0.0, y = 0.0, z = 0.0, inv = 0.0, g4[4] = {0.0, 0.0, 0.0, 0.0}, dg4[4] = {0.0, 0.0, 0.0, 0.0};
            double px = 0.0, py = 0.0, pz = 0.0;
            if (r2 < rcr2) {
                inv = rsqrt(r2);
                const double r = r2 * inv;
                x = dx * inv; y = dy * inv; z = dz * inv;
                if (pass == 0) {  // radial descriptors: sum_n Fd_n g'_n(r) u
                    double f[KMAX], df[KMAX];
                    nep_basis<KMAX>(r * ircr, ircr, sp.kr, f, df);
                    const double *c = cRb + (size_t)J * kNepMaxN * KMAX;
                    double sr = 0.0;
#pragma unroll
                    for (int nn = 0; nn < kNepMaxN; ++nn) {
                        double dg = 0.0;
#pragma unroll
                        for (int b = 0; b < KMAX; ++b) dg += c[nn * KMAX + b] * df[b];
                        sr += FdR[nn] * dg;
                    }
                    px = sr * x; py = sr * y; pz = sr * z;
                }
                if (r2 < rca2) {
                    double f[KMAX], df[KMAX];
                    nep_basis<KMAX>(r * irca, irca, sp.ka, f, df);
#pragma unroll
                    for (int c4 = 0; c4 < 4; ++c4) {
                        const double *c = cAb + ((size_t)J * kNepMaxN + 4 * pass + c4) * KMAX;
                        double g = 0.0, dg = 0.0;
#pragma unroll
                        for (int b = 0; b < KMAX; ++b) { g += c[b] * f[b]; dg += c[b] * df[b]; }
                        g4[c4] = g;
                        dg4[c4] = dg;
                    }
                }
            }
            const double inA = r2 < rca2 ? 1.0 : 0.0;
#pragma unroll
            for (int t = 0; t < 4; ++t) {
                const int src = (q + t) & 3;
                const double gs = t == 0 ? sel4(g4, q) : shf(sel4(g4, (q - t) & 3), src);
                const double dgs = t == 0 ? sel4(dg4, q) : shf(sel4(dg4, (q - t) & 3), src);
                const double xs = t == 0 ? x : shf(x, src), ys = t == 0 ? y : shf(y, src), zs = t == 0 ? z : shf(z, src);
                const double is = t == 0 ? inv : shf(inv, src), as = t == 0 ? inA : shf(inA, src);
                double cx = 0.0, cy = 0.0, cz = 0.0;
                if (own && as != 0.0) {
                    double m[kNepC];
                    nep_monomials(xs, ys, zs, m);  // only the monomials of degree <= 3 are read below
                    double gl[4][3];
                    nep_poly_grad(G, m, gl);
                    double phi = G[0], ug = 0.0, gx = 0.0, gy = 0.0, gz = 0.0;
#pragma unroll
                    for (int l = 0; l < 4; ++l) {  // u . grad phi_l = l phi_l (Euler)
                        const double tt = xs * gl[l][0] + ys * gl[l][1] + zs * gl[l][2];
                        ug += tt;
                        phi += tt * (1.0 / (l + 1));
                        gx += gl[l][0]; gy += gl[l][1]; gz += gl[l][2];
                    }
                    const double gi = gs * is, dphi = dgs * phi;
                    cx = dphi * xs + gi * (gx - ug * xs);
                    cy = dphi * ys + gi * (gy - ug * ys);
                    cz = dphi * zs + gi * (gz - ug * zs);
                }
                // back to the row's lane: in step t this lane's row was evaluated by lane q - t
                const int ev = (q - t) & 3;
                px += t == 0 ? cx : shf(cx, ev);
                py += t == 0 ? cy : shf(cy, ev);
                pz += t == 0 ? cz : shf(cz, ev);
            }
            if (kk < cnt) {
                double *o = part + (size_t)(kk * 3) * d.Npad;
                if (pass) { px += o[0]; py += o[d.Npad]; pz += o[2 * (size_t)d.Npad]; }
                o[0] = px; o[d.Npad] = py; o[2 * (size_t)d.Npad] = pz;
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
    const NepShape sp = nep_shape(d.pot);
    const int kmax = (int)(d.pot[4] > d.pot[5] ? d.pot[4] : d.pot[5]), KM = kmax <= 4 ? 4 : kmax <= 8 ? 8 : 12;
    const size_t smem = ((size_t)((sp.T * nep_net_size(sp) + 1) & ~1) + 2 * (size_t)sp.T * sp.T * kNepMaxN * KM) * sizeof(double);
    static bool attr_set = false;
    if (!attr_set) {
        cudaFuncSetAttribute(nep_partial_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
        cudaFuncSetAttribute(nep_partial_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
        cudaFuncSetAttribute(nep_partial_kernel<12>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
        attr_set = true;
    }
    if (kmax <= 4) nep_partial_kernel<4><<<grid, kNepThreads, smem, st>>>(d, p_lo);
    else if (kmax <= 8) nep_partial_kernel<8><<<grid, kNepThreads, smem, st>>>(d, p_lo);
    else nep_partial_kernel<12><<<grid, kNepThreads, smem, st>>>(d, p_lo);
    launch_pair_forces_manybody(d, p_lo, st);
}

}  // namespace cfn

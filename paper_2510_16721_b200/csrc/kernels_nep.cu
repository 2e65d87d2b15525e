// kernels_nep.cu -- K2, pass 1, for the NEP-shaped potential CFNEB_POT_NEP (include/cfneb.h): the descriptor network of
// kernels_dn.cu widened to the shape and cost of the paper's force field proper ("NEP-trained force field";
// its evaluation is the 10^6 atom-steps per second the paper quotes): separate radial and angular cut-offs,
// two atom types with type-pair expansion coefficients, basis sizes and descriptor counts as parameters, Legendre
// orders up to 4, one network of up to 64 neurons per type.  Seeded weights (the trained ones are not available):
// cost and data flow, no physics.  It enters the path through the partial forces p^ij = dU_i/dr^ij of Eq. 5; pass 2
// (f^ij = p^ij - p^ji, F_i, virial of Eq. 8) of the angular part is the kernel the other many-body potentials use
// (kernels_sw.cu), the radial part is formed pair by pair.
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
// Work split: four launches (launch_force_nep).
//  1. nep_radial_desc_kernel, one atom per thread over all live rows: q_n through the basis sums per neighbour type.
//  2. nep_partial_kernel, FOUR LANES PER ATOM, over the rows that can lie inside rc_a only (nep_angular_rows): lane q of
//     a quad owns the angular channels n = q, q + 4 and a quarter of the neurons.  The list is walked four rows at a
//     time, ONE ROW PER LANE: a lane forms the pair vector, the angular basis and the expansions g_n of its row once,
//     then the rows go round the quad by shuffles and every lane adds each row to the 35 moments of its own channel
//     (registers); the moments are parked in a scratch array (one 280-byte column per atom and channel), the network
//     runs on the fp64 tensor cores (a warp's eight quads are the eight rows of an m8n8k4 fragment; the quad's
//     descriptors side by side in shared memory are the A operand), and a second walk of the same shape evaluates
//     phi_n(u) = sum_c G_nc u^c and its gradient per channel and hands the three components back to the row's lane,
//     which writes the angular partial force once.  Network weights and angular expansion coefficients sit in shared
//     memory.  The radial descriptors act on the forces through w_i[J][k] = sum_n dU_i/dq_n cR[I][J][n][k], written
//     out per atom.
//  3. nep_radial_pair_kernel, one atom per thread over all live rows: the radial part of Eq. 5 pair by pair from
//     w_i[J] + w_j[I]; F_i and the virial partials of that part.
//  4. pass 2 of the angular partial forces over the angular rows (kernels_sw.cu), added to F_i.
// No per-thread environment array, hence no limit on the atoms inside the cut-offs but the list capacity.  The type of
// an atom rides in the fourth double of its position sector (positions_kernel).
#include "cfneb_internal.cuh"
#include "nep_poly.cuh"
#include "trig01.cuh"

namespace cfn {

constexpr int kNepMaxN = 8, kNepMaxH = 64, kNepMaxL = 4, kNepMaxD = kNepMaxN + kNepMaxN * kNepMaxL;
constexpr int kNepThreads = 128;  // 32 atoms x 4 lanes
#ifndef CFNEB_NEP_BLOCKS
#define CFNEB_NEP_BLOCKS 3
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
// layout of Dev::dn_w for this potential: per type [W0t Dp*HS | b0 Hp | W1 Hp] (first layer transposed to [d][mu];
// neurons and descriptors zero-padded to multiples of eight, Hp and Dp, rows HS = Hp + 4 doubles apart so that the
// tensor-core fragment loads of the quad kernel fall on distinct banks; copied to shared memory as it is), then
// cR [T][T][nr][kr], then cA [T][T][na][ka]
__host__ __device__ inline int nep_hp(const NepShape &s) { return (s.H + 7) & ~7; }
__host__ __device__ inline int nep_dp(const NepShape &s) { return (s.D + 7) & ~7; }
__host__ __device__ inline int nep_hs(const NepShape &s) { return nep_hp(s) + 4; }
__host__ __device__ inline int nep_net_size(const NepShape &s) { return nep_dp(s) * nep_hs(s) + 2 * nep_hp(s); }
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

// D = A B + D on the fp64 tensor cores, m8n8k4: lane l holds A[l >> 2][l & 3], B[l & 3][l >> 2], D[l >> 2][2 (l & 3) + {0, 1}]
__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

__device__ __forceinline__ const double4 *Rc_of(const Dev &d, int slot) { return d.Rc + (size_t)slot * d.Npad; }

// One atom per thread over all live rows of its list, the loads software-pipelined with NO register rotation (a
// move of a register whose load is in flight waits for the load: the rotating version of this walk spent a third
// of its stall samples on such a move).  The loop is unrolled over the four entry registers: in stage u (row k + u)
// the sector of row k + u + 1 is requested through the entry that was loaded three stages ago, the entry register of
// this row is reloaded for row k + u + 4, and the list row twelve ahead is pulled into L2.
// body(k, j, rj, dx, dy, dz, r2) for the rows k < cnt of this thread (rj.w = type of the neighbour j).
// (Requesting w_j of the next row a stage ahead in nep_radial_pair_kernel, into registers or into L1, measured slower.)
template <class Body>
__device__ __forceinline__ void nep_walk_rows(const Dev &d, const uint32_t *lp, const double4 *Rc, const double4 &ri,
                                              const double *sh, int cnt, Body body) {
    if (cnt <= 0) return;
    const int last = cnt - 1;
    uint32_t e[4];
    double4 s[2];
#pragma unroll
    for (int u = 0; u < 4; ++u) e[u] = lp[(size_t)min(u, last) * d.Npad];
    s[0] = Rc[e[0] & kIdxMask];
    auto stage = [&](int k, uint32_t &ecur, uint32_t enext, const double4 &scur, double4 &snext) {
        snext = Rc[enext & kIdxMask];
        const uint32_t code = ecur >> kShiftBits, j = ecur & kIdxMask;
        ecur = lp[(size_t)min(k + 4, last) * d.Npad];
        asm volatile("prefetch.global.L2 [%0];" ::"l"(lp + (size_t)min(k + 12, last) * d.Npad));
        double dx = scur.x - ri.x, dy = scur.y - ri.y, dz = scur.z - ri.z;
        if (code != kCodeCenter) {
            const double n0 = (double)((int)(code & 7u) - 4), n1 = (double)((int)((code >> 3) & 7u) - 4),
                         n2 = (double)((int)((code >> 6) & 7u) - 4);
            dx += n0 * sh[0] + n1 * sh[3] + n2 * sh[6];
            dy += n0 * sh[1] + n1 * sh[4] + n2 * sh[7];
            dz += n0 * sh[2] + n1 * sh[5] + n2 * sh[8];
        }
        body(k, j, scur, dx, dy, dz, dx * dx + dy * dy + dz * dz);
    };
    for (int k = 0; k < cnt; k += 4) {
        stage(k, e[0], e[1], s[0], s[1]);
        if (k + 1 >= cnt) break;
        stage(k + 1, e[1], e[2], s[1], s[0]);
        if (k + 2 >= cnt) break;
        stage(k + 2, e[2], e[3], s[0], s[1]);
        if (k + 3 >= cnt) break;
        stage(k + 3, e[3], e[0], s[1], s[0]);
    }
}

constexpr int kNepRadialThreads = 128;
#ifndef CFNEB_NEP_RADIAL_BLOCKS
#define CFNEB_NEP_RADIAL_BLOCKS 4
#endif

// Radial descriptors q_n = sum_j sum_k cR[I][J][n][k] f_k(r_ij; rc_r) -> Dev::nep_q.  One atom per thread; the sum
// over the environment is taken per neighbour type on the basis functions, B[J][k] = sum_{j of type J} f_k(r_ij),
// and the coefficients are applied once per atom (k_r adds per row instead of n_r k_r multiply-adds).
template <int KMAX, int NT>
__global__ void __launch_bounds__(kNepRadialThreads, CFNEB_NEP_RADIAL_BLOCKS) nep_radial_desc_kernel(Dev d, int p_lo) {
    int p;
    if (!image_of(blockIdx.y, p_lo, d.ctl->P, p)) return;
    const int slot = d.order[p];
    __shared__ double sh[9];
    if (threadIdx.x < 9) sh[threadIdx.x] = d.geom[slot].h[threadIdx.x];
    __syncthreads();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= d.N) return;
    const NepShape sp = nep_shape(d.pot);
    const double rcr = d.pot[0], rcr2 = rcr * rcr, ircr = 1.0 / rcr;
    const double4 *Rc = Rc_of(d, slot);
    const double4 ri = Rc[i];
    double B[NT][KMAX];
#pragma unroll
    for (int J = 0; J < NT; ++J)
#pragma unroll
        for (int k = 0; k < KMAX; ++k) B[J][k] = 0.0;
    nep_walk_rows(d, d.nbr_list + (size_t)slot * d.cap * d.Npad + i, Rc, ri, sh, live_rows(d, slot, i),
                  [&](int, uint32_t, const double4 &rj, double, double, double, double r2) {
        if (r2 < rcr2) {
            // B[J][k] accumulates fc T_k (f_k = 1/2 (T_k + 1) fc is put together once per atom below); T_k runs to
            // KMAX with no guard: |x| <= 1 and the entries beyond k_r are never read
            const double t = r2 * rsqrt_nr(r2) * ircr, fc = 0.5 + 0.5 * cospi01(t);
            const double x = 2.0 * (t - 1.0) * (t - 1.0) - 1.0, x2 = 2.0 * x;
            const double m1 = NT > 1 ? rj.w * fc : 0.0, m0 = fc - m1;  // type of the neighbour as a weight
            double Tm = 1.0, Tk = x;
#pragma unroll
            for (int k = 0; k < KMAX; ++k) {
                const double Tv = k == 0 ? 1.0 : Tk;
                B[0][k] = fma(m0, Tv, B[0][k]);
                if (NT > 1) B[NT - 1][k] = fma(m1, Tv, B[NT - 1][k]);
                if (k >= 1) { const double Tn = fma(x2, Tk, -Tm); Tm = Tk; Tk = Tn; }
            }
        }
    });
    const int I = (int)ri.w;
    const double *cR = d.dn_w + sp.T * nep_net_size(sp) + (size_t)I * sp.T * sp.nr * sp.kr;  // [J][n][k]
    double *qscr = d.nep_q + (size_t)slot * kNepMaxN * d.Npad + i;
    for (int n = 0; n < sp.nr; ++n) {
        double qn = 0.0;
#pragma unroll
        for (int J = 0; J < NT; ++J)
#pragma unroll
            for (int k = 0; k < KMAX; ++k)
                if (k < sp.kr) qn = fma(cR[(J * sp.nr + n) * sp.kr + k], B[J][k] + B[J][0], qn);  // B[J][0] = sum fc
        qscr[(size_t)n * d.Npad] = 0.5 * qn;
    }
}

// Radial part of the forces, pair by pair (no partial forces stored): p^ij = [sum_k w_i[J][k] f_k'(r_ij)] u_ij with
// w_i[J][k] = sum_n dU_i/dq_n cR[I][J][n][k] (formed once per atom by the quad kernel, Dev::nep_w), and the mirror term
// of Eq. 5 is the same expression with j's coefficients for i's type, so
//   f^ij = p^ij - p^ji = [sum_k (w_i[J][k] + w_j[I][k]) f_k'(r_ij)] u_ij
// needs one 8 k_r-byte gather per row instead of a stored partial force and its mirror.  One atom per thread over all
// live rows; writes F_i and the virial partials of this part, the angular part is added by pass 2 (kernels_sw.cu).
template <int KMAX, int NT>
__global__ void __launch_bounds__(kNepRadialThreads, CFNEB_NEP_RADIAL_BLOCKS) nep_radial_pair_kernel(Dev d, int p_lo) {
    int p;
    if (!image_of(blockIdx.y, p_lo, d.ctl->P, p)) return;
    const int slot = d.order[p];
    __shared__ double sh[9];
    __shared__ double red[32 * 6];
    __shared__ double2 sWi[NT * (KMAX / 2) * kNepRadialThreads];  // this thread's w_i[J][k], two k per entry, thread-minor
    if (threadIdx.x < 9) sh[threadIdx.x] = d.geom[slot].h[threadIdx.x];
    __syncthreads();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = i < d.N;
    const NepShape sp = nep_shape(d.pot);
    const double rcr = d.pot[0], rcr2 = rcr * rcr, ircr = 1.0 / rcr;
    const double4 *Rc = Rc_of(d, slot);
    const double *wv = d.nep_w + (size_t)slot * d.Npad * (NT * KMAX);  // wv[(j * NT + J) * KMAX + k]
    double fx = 0.0, fy = 0.0, fz = 0.0, vxx = 0.0, vyy = 0.0, vzz = 0.0, vxy = 0.0, vxz = 0.0, vyz = 0.0;
    if (valid) {
        const double4 ri = Rc[i];
        const int I = (int)ri.w;
#pragma unroll
        for (int t = 0; t < NT * (KMAX / 2); ++t)
            sWi[t * kNepRadialThreads + threadIdx.x] = reinterpret_cast<const double2 *>(wv + (size_t)i * NT * KMAX)[t];
        nep_walk_rows(d, d.nbr_list + (size_t)slot * d.cap * d.Npad + i, Rc, ri, sh, live_rows(d, slot, i),
                      [&](int, uint32_t j, const double4 &rj, double dx, double dy, double dz, double r2) {
            if (r2 < rcr2) {
                double2 wjk[KMAX / 2];
#pragma unroll
                for (int t = 0; t < KMAX / 2; ++t) wjk[t] = reinterpret_cast<const double2 *>(wv + ((size_t)j * NT + I) * KMAX)[t];
                const double inv = rsqrt_nr(r2);
                const double2 *wi = sWi + (NT > 1 ? (int)rj.w : 0) * (KMAX / 2) * kNepRadialThreads + threadIdx.x;
                // sum_k W_k f_k' with W_k = w_i[J][k] + w_j[I][k] and f_k' = 1/2 T_k' x' fc + 1/2 (T_k + 1) fc':
                //   = 1/2 x' fc sum_k W_k T_k' + 1/2 fc' (sum_k W_k T_k + sum_k W_k); W_k = 0 beyond k_r, no guard
                const double t = r2 * inv * ircr;
                double sn, cs;
                sincospi01(t, sn, cs);
                const double fc = 0.5 + 0.5 * cs, dfc = -0.5 * sn * (3.14159265358979323846 * ircr);
                const double x = 2.0 * (t - 1.0) * (t - 1.0) - 1.0, x2 = 2.0 * x, dx_dr = 4.0 * (t - 1.0) * ircr;
                double Tm = 1.0, Tk = x, dTm = 0.0, dTk = 1.0, sT = 0.0, sdT = 0.0, sW = 0.0;
#pragma unroll
                for (int k = 0; k < KMAX; ++k) {
                    const double2 a = wi[(k >> 1) * kNepRadialThreads];
                    const double W = (k & 1) ? a.y + wjk[k >> 1].y : a.x + wjk[k >> 1].x;
                    sW += W;
                    if (k == 0) { sT = W; continue; }
                    sT = fma(W, Tk, sT);
                    sdT = fma(W, dTk, sdT);
                    const double Tn = fma(x2, Tk, -Tm), dTn = fma(x2, dTk, fma(2.0, Tk, -dTm));
                    Tm = Tk; Tk = Tn; dTm = dTk; dTk = dTn;
                }
                const double sr = 0.5 * (dx_dr * fc * sdT + dfc * (sT + sW)) * inv;
                const double gx = sr * dx, gy = sr * dy, gz = sr * dz;  // f^ij of Eq. 5, radial part
                fx += gx; fy += gy; fz += gz;
                vxx = fma(dx, gx, vxx); vyy = fma(dy, gy, vyy); vzz = fma(dz, gz, vzz);  // Eq. 8 (central: symmetric)
                vxy = fma(dx, gy, vxy); vxz = fma(dx, gz, vxz); vyz = fma(dy, gz, vyz);
            }
        });
        double *F = d.F + (size_t)slot * 3 * d.Npad;
        F[i] = fx; F[d.Npad + i] = fy; F[2 * (size_t)d.Npad + i] = fz;
    }
    double out6[6] = {-0.5 * vxx, -0.5 * vyy, -0.5 * vzz, -0.5 * vxy, -0.5 * vxz, -0.5 * vyz};
    block_sum<6>(out6, red);
    if (threadIdx.x == 0) {
        double *out = d.part_force + ((size_t)slot * d.nblk_force + blockIdx.x) * kNForcePart;
        out[0] = 0.0;
#pragma unroll
        for (int n = 0; n < 6; ++n) out[1 + n] = out6[n];
        out[8] = 0.0;
    }
}

// KMAX: basis functions held per row (the smallest of 4, 8, 12 that covers k_r and k_a): the loops over them are
// unrolled so that the basis stays in registers.
template <int KMAX>
__global__ void __launch_bounds__(kNepThreads, CFNEB_NEP_BLOCKS) nep_partial_kernel(Dev d, int p_lo) {
    int p;
    if (!image_of(blockIdx.y, p_lo, d.ctl->P, p)) return;
    const int slot = d.order[p];
    extern __shared__ __align__(16) double sW[];  // all weights of the potential
    __shared__ double sh[9];
    __shared__ double red[64];
    __shared__ double sQ[(kNepThreads / 4) * (kNepMaxD + 1)];  // descriptors, then their gradients, one row per quad
    const NepShape sp = nep_shape(d.pot);
    const int nNet = sp.T * nep_net_size(sp);  // offset of the expansion coefficients in Dev::dn_w
    const int Hp = nep_hp(sp), netp = nep_net_size(sp);
    if (threadIdx.x < 9) sh[threadIdx.x] = d.geom[slot].h[threadIdx.x];
    // the network weights are not needed before the first walk is over: asynchronous copy (16 bytes per request;
    // nNet is even and both sides are 16-byte aligned), waited for in front of the network
    for (int t = 2 * threadIdx.x; t < nNet; t += 2 * blockDim.x)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(sW + t)), "l"(d.dn_w + t));
    asm volatile("cp.async.commit_group;");
    // angular expansion coefficients zero-padded to [T][T][8][KMAX]: the loops over channels and basis functions then
    // run to their compile-time bounds with no guards, and a row of coefficients is KMAX aligned doubles
    double *cAp = sW + ((nNet + 1) & ~1);
    for (int t = threadIdx.x; t < sp.T * sp.T * kNepMaxN * KMAX; t += blockDim.x) {
        const int b = t % KMAX, nn = (t / KMAX) % kNepMaxN, IJ = t / (KMAX * kNepMaxN);
        cAp[t] = (nn < sp.na && b < sp.ka) ? d.dn_w[nNet + sp.T * sp.T * sp.nr * sp.kr + (IJ * sp.na + nn) * sp.ka + b] : 0.0;
    }
    __syncthreads();
    const int q = threadIdx.x & 3;                                     // lane of the quad
    const int i = blockIdx.x * (kNepThreads / 4) + (threadIdx.x >> 2);  // atom of the quad
    const bool valid = i < d.N;
    const int ic = valid ? i : 0;
    const unsigned quad_mask = 0xffffffffu;  // see cnt_w below
    const double rca = d.pot[1], rca2 = rca * rca, irca = 1.0 / rca;
    const double4 ri = Rc_of(d, slot)[ic];
    const int I = (int)ri.w;
    const double *b0 = sW + I * netp + nep_dp(sp) * nep_hs(sp), *W1 = b0 + Hp;  // of this atom's type
    const double *cAb = cAp + (size_t)I * sp.T * kNepMaxN * KMAX;
    const double4 *Rc = Rc_of(d, slot);
    const uint32_t *lp = d.nbr_list + (size_t)slot * d.cap * d.Npad + ic;
    double *part = d.part + (size_t)slot * d.cap * 3 * d.Npad + ic;  // part[(k * 3 + m) * Npad]
    double *scr = d.nep_S + ((size_t)slot * sp.na * kNepC) * d.Npad + ic;  // scr[(n * kNepC + c) * Npad]
    double *qscr = d.nep_q + (size_t)slot * kNepMaxN * d.Npad + ic;       // qscr[n * Npad]
    const int cnt = valid ? nep_angular_rows(d, slot, ic) : 0;  // rows past it cannot be inside rc_a
    // every loop over list rows runs to the longest list of the warp (rows past a quad's own count are skipped by
    // `kk < cnt`): all 32 lanes reach every shuffle, so the shuffles take the full mask
    const int cnt_w = __reduce_max_sync(0xffffffffu, cnt);

    // The rows of a lane (kk = q, q + 4, ...) are software-pipelined: the list entry two rows ahead and the neighbour's
    // sector and type one row ahead are in flight while a row is evaluated (two resident warps per scheduler cannot
    // hide the two dependent loads otherwise).  Rows past the end stand in with the atom itself and are never used.
    uint32_t e_nn, e_n;
    double4 rj_n;
    auto walk_begin = [&]() {
        e_n = q < cnt ? lp[(size_t)q * d.Npad] : (uint32_t)ic | (kCodeCenter << kShiftBits);
        e_nn = q + 4 < cnt ? lp[(size_t)(q + 4) * d.Npad] : e_n;
        rj_n = Rc[e_n & kIdxMask];
    };
    auto pair_vec = [&](int k, int &J, double &dx, double &dy, double &dz) {  // row k of this lane; advances the pipeline
        const uint32_t code = e_n >> kShiftBits;
        const double4 rj = rj_n;
        J = (int)rj.w;  // positions_kernel puts the type there
        e_n = e_nn;
        e_nn = k + 8 < cnt ? lp[(size_t)(k + 8) * d.Npad] : e_n;
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

    const int base_lane = (threadIdx.x & 31) & ~3;
    auto shf = [&](double v, int src) { return __shfl_sync(quad_mask, v, base_lane + src); };
    auto quad_sum = [&](double v) {
        v += __shfl_xor_sync(quad_mask, v, 1);
        return v + __shfl_xor_sync(quad_mask, v, 2);
    };

    // ---- walk 1: the list is taken four rows at a time, ONE ROW PER LANE: the lane forms the pair vector, the radial
    // basis and the expansions g_n of its row (nothing of that is done four times), then the rows go round the quad
    // (step t: lane q takes the row of lane q + t) and each lane adds every row to the moments of its own channel ----
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
            if (r2 < rca2) {
                const double inv = rsqrt_nr(r2), r = r2 * inv;
                x = dx * inv; y = dy * inv; z = dz * inv;
                double f[KMAX], df[KMAX];
                nep_basis<KMAX>(r * irca, irca, sp.ka, f, df);
#pragma unroll
                for (int c4 = 0; c4 < 4; ++c4) {  // g4[t]: the channel that lane q - t owns, read by it in step t
                    const double *c = cAb + ((size_t)J * kNepMaxN + 4 * pass + ((q - c4) & 3)) * KMAX;
                    double g = 0.0;
#pragma unroll
                    for (int b = 0; b < KMAX; ++b) g += c[b] * f[b];
                    g4[c4] = g;
                }
            }
            const double inA = r2 < rca2 ? 1.0 : 0.0;
#pragma unroll
            for (int t = 0; t < 4; ++t) {
                const int src = (q + t) & 3;
                // step t: this lane reads from lane src = q + t the g of its own channel, which that lane holds as
                // its g4[t] (channel (src - t) & 3 = q)
                const double gs = t == 0 ? g4[0] : shf(g4[t], src);
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
    // ---- the network, on the fp64 tensor cores: a warp is eight quads = eight atoms = the eight rows of an m8n8k4
    // fragment.  Forward z[atom][mu] = sum_d q[atom][d] W0[mu][d]: lane q of quad g supplies A[g][q] = q_{k0 + q} of its
    // atom, loads B[q][g] = W0t[k0 + q][8 t + g], and receives C[g][2 q], C[g][2 q + 1]: the neurons 8 t + 2 q, + 1 of
    // its own atom, eight per lane.  The weights are per atom type and a warp holds atoms of both: each type's matrix is
    // applied with the rows of the other type's atoms zeroed, into the same accumulators.  Backward
    // dU/dq_d = sum_mu g_mu W0[mu][d] the same way with the lane's own neurons as the A operand (k-step (t, h) takes
    // neuron 8 t + 2 q + h from lane q).  Padded neurons (b0 = W0 = W1 = 0) and padded descriptors contribute nothing. ----
    double ui = 0.0;
    double FdA[2][kNepMaxL] = {};
    asm volatile("cp.async.wait_all;");
    __syncthreads();  // the weights of the other threads' requests
    {
        const int Dp = nep_dp(sp), HS = nep_hs(sp), ntile = Hp >> 3, g = (threadIdx.x & 31) >> 2;
        double zt[kNepMaxH / 4];  // zt[2 t + c]: neuron 8 t + 2 q + c
#pragma unroll
        for (int t = 0; t < kNepMaxH / 8; ++t) {
            zt[2 * t] = t < ntile ? -b0[8 * t + 2 * q] : 0.0;
            zt[2 * t + 1] = t < ntile ? -b0[8 * t + 2 * q + 1] : 0.0;
        }
        // the descriptors of the quad's atom side by side in shared memory, zero beyond D
        double *sq = sQ + (threadIdx.x >> 2) * (kNepMaxD + 1);  // odd stride: the quads of a warp on distinct banks
        for (int n = q; n < Dp; n += 4) sq[n] = (n < sp.nr && valid) ? qscr[(size_t)n * d.Npad] : 0.0;
        __syncwarp();
#pragma unroll
        for (int hh = 0; hh < 2; ++hh)
#pragma unroll
            for (int ll = 0; ll < kNepMaxL; ++ll)
                if (q + 4 * hh < sp.na && ll < sp.L) sq[sp.nr + (q + 4 * hh) * sp.L + ll] = qA[hh][ll];
        __syncwarp();
        for (int T2 = 0; T2 < sp.T; ++T2) {
            const double *Wt = sW + T2 * netp;
            for (int k0 = 0; k0 < Dp; k0 += 4) {
                const double a = I == T2 ? sq[k0 + q] : 0.0;
                const double *brow = Wt + (k0 + q) * HS + g;
#pragma unroll
                for (int t = 0; t < kNepMaxH / 8; ++t) {
                    if (t >= ntile) break;
                    dmma884(zt[2 * t], zt[2 * t + 1], a, brow[8 * t]);
                }
            }
        }
        __syncwarp();
        double gmu[kNepMaxH / 4];
#pragma unroll
        for (int t = 0; t < kNepMaxH / 4; ++t) {
            gmu[t] = 0.0;
            if ((t >> 1) < ntile) {
                const double th = tanh(zt[t]), w1 = W1[8 * (t >> 1) + 2 * q + (t & 1)];
                ui = fma(w1, th, ui);
                gmu[t] = w1 * (1.0 - th * th);
            }
        }
        // dU/dq_d (the radial ones go on to nep_radial_pair_kernel as w_i, the angular ones back to their owners)
        for (int n0 = 0; n0 < Dp; n0 += 8) {
            double c0 = 0.0, c1 = 0.0;
            for (int T2 = 0; T2 < sp.T; ++T2) {
                const double *bcol = sW + T2 * netp + (n0 + g) * HS + 2 * q;
#pragma unroll
                for (int t = 0; t < kNepMaxH / 8; ++t) {
                    if (t >= ntile) break;
                    dmma884(c0, c1, I == T2 ? gmu[2 * t] : 0.0, bcol[8 * t]);
                    dmma884(c0, c1, I == T2 ? gmu[2 * t + 1] : 0.0, bcol[8 * t + 1]);
                }
            }
            sq[n0 + 2 * q] = c0;
            sq[n0 + 2 * q + 1] = c1;
        }
        __syncwarp();
        // the radial descriptors act on the forces through w_i[J][k] = sum_n dU/dq_n cR[I][J][n][k] alone
        // (nep_radial_pair_kernel): the quad forms the T KR of them, zero beyond k_r
        if (valid) {
            const int KR = d.nep_kr_pad;
            const double *cR = d.dn_w + nNet + (size_t)I * sp.T * sp.nr * sp.kr;  // [J][n][k]
            double *wv = d.nep_w + ((size_t)slot * d.Npad + ic) * (sp.T * KR);
            for (int t = q; t < sp.T * KR; t += 4) {
                const int J = t / KR, k = t % KR;
                double w = 0.0;
                if (k < sp.kr)
                    for (int n = 0; n < sp.nr; ++n) w = fma(sq[n], cR[(J * sp.nr + n) * sp.kr + k], w);
                wv[t] = w;
            }
        }
#pragma unroll
        for (int hh = 0; hh < 2; ++hh)
#pragma unroll
            for (int ll = 0; ll < kNepMaxL; ++ll)
                if (q + 4 * hh < sp.na && ll < sp.L) FdA[hh][ll] = sq[sp.nr + (q + 4 * hh) * sp.L + ll];
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
            if (r2 < rca2) {
                inv = rsqrt_nr(r2);
                const double r = r2 * inv;
                x = dx * inv; y = dy * inv; z = dz * inv;
                double f[KMAX], df[KMAX];
                nep_basis<KMAX>(r * irca, irca, sp.ka, f, df);
#pragma unroll
                for (int c4 = 0; c4 < 4; ++c4) {  // g4[t], dg4[t]: the channel of lane q - t (walk 1)
                    const double *c = cAb + ((size_t)J * kNepMaxN + 4 * pass + ((q - c4) & 3)) * KMAX;
                    double g = 0.0, dg = 0.0;
#pragma unroll
                    for (int b = 0; b < KMAX; ++b) { g += c[b] * f[b]; dg += c[b] * df[b]; }
                    g4[c4] = g;
                    dg4[c4] = dg;
                }
            }
            const double inA = r2 < rca2 ? 1.0 : 0.0;
#pragma unroll
            for (int t = 0; t < 4; ++t) {
                const int src = (q + t) & 3;
                const double gs = t == 0 ? g4[0] : shf(g4[t], src);
                const double dgs = t == 0 ? dg4[0] : shf(dg4[t], src);
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
int nep_kr_padded(const double *pot) { const int kr = (int)pot[4]; return kr <= 4 ? 4 : kr <= 8 ? 8 : 12; }

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
    const int Hp = nep_hp(s);
    for (int I = 0; I < s.T; ++I) {  // stream order: W0[mu][d], b0[mu], W1[mu]
        double *net = w + (size_t)I * nep_net_size(s);
        for (int t = 0; t < nep_net_size(s); ++t) net[t] = 0.0;
        const int HS = nep_hs(s), Dp = nep_dp(s);
        for (int t = 0; t < s.H * s.D; ++t) net[(t % s.D) * HS + t / s.D] = next() * ((t % s.D) < s.nr ? 0.04 : 0.004);
        for (int t = 0; t < s.H; ++t) net[Dp * HS + t] = 0.5 * next();
        for (int t = 0; t < s.H; ++t) net[Dp * HS + Hp + t] = next();
    }
    double *c = w + (size_t)s.T * nep_net_size(s);
    const int nc = s.T * s.T * (s.nr * s.kr + s.na * s.ka);
    for (int t = 0; t < nc; ++t) c[t] = next();
}

template <int KMAX>
static void launch_nep_radial(const Dev &d, int p_lo, dim3 grid, bool force, cudaStream_t st) {
    const int nt = (int)d.pot[8];
    if (force) {
        if (nt <= 1) nep_radial_pair_kernel<KMAX, 1><<<grid, kNepRadialThreads, 0, st>>>(d, p_lo);
        else nep_radial_pair_kernel<KMAX, 2><<<grid, kNepRadialThreads, 0, st>>>(d, p_lo);
    } else {
        if (nt <= 1) nep_radial_desc_kernel<KMAX, 1><<<grid, kNepRadialThreads, 0, st>>>(d, p_lo);
        else nep_radial_desc_kernel<KMAX, 2><<<grid, kNepRadialThreads, 0, st>>>(d, p_lo);
    }
}

// The quad kernel's dynamic shared memory (network weights + expansion coefficients) passes the 48 KB default at the
// larger shapes (H = 64, D = 40, two types: 48.6 KB): opt in.  The attribute belongs to the (function, device) pair, so
// this runs in every cfneb_create with the handle's device current -- not once per process -- and its failure is an
// error of that call.
cudaError_t prepare_nep_kernels() {
    cudaError_t e = cudaFuncSetAttribute(nep_partial_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(nep_partial_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(nep_partial_kernel<12>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    return e;
}

// Four launches: radial descriptors (one atom per thread, all live rows), the quad kernel (angular rows, network,
// angular partial forces), the radial forces pair by pair (one atom per thread, all live rows), pass 2 of the angular
// partial forces over the angular rows (kernels_sw.cu), which adds to F and to the virial partials.
void launch_force_nep(const Dev &d, int p_lo, cudaStream_t st) {
    const int nimg = images_in_grid(d.S, p_lo);
    if (nimg <= 0) return;
    const NepShape sp = nep_shape(d.pot);
    const dim3 grid(d.nblk_force, nimg), grid_r((d.N + kNepRadialThreads - 1) / kNepRadialThreads, nimg);
    const int KR = sp.kr <= 4 ? 4 : sp.kr <= 8 ? 8 : 12, KA = sp.ka <= 4 ? 4 : sp.ka <= 8 ? 8 : 12;
    const size_t smem = ((size_t)((sp.T * nep_net_size(sp) + 1) & ~1) + (size_t)sp.T * sp.T * kNepMaxN * KA) * sizeof(double);
    for (int force = 0; force < 2; ++force) {
        if (KR == 4) launch_nep_radial<4>(d, p_lo, grid_r, force, st);
        else if (KR == 8) launch_nep_radial<8>(d, p_lo, grid_r, force, st);
        else launch_nep_radial<12>(d, p_lo, grid_r, force, st);
        if (force) break;
        if (KA == 4) nep_partial_kernel<4><<<grid, kNepThreads, smem, st>>>(d, p_lo);
        else if (KA == 8) nep_partial_kernel<8><<<grid, kNepThreads, smem, st>>>(d, p_lo);
        else nep_partial_kernel<12><<<grid, kNepThreads, smem, st>>>(d, p_lo);
    }
    launch_pair_forces_manybody(d, p_lo, st);
}

}  // namespace cfn

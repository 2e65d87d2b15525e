// kernels_force.cu -- K2: batched images x atoms energy / force / virial (Eq. 4, 5, 8).
//
//   r^ij = R_j - R_i + n h            (r^ij = r^j - r^i; n = periodic shift of the list entry)
//   F_i  = sum_j f^ij,  f^ij = fmag(r) r^ij / r   (force on i due to j, Eq. 5 applied to the U_i below)
//   V_mn = -1/2 sum_i sum_j r^ij_m f^ij_n          (Eq. 7-8)
//   E    = sum_i U_i                                (Eq. 4)
//
// Potentials (BASELINE.json configs; O3, reading A21):
//   LJ shifted-force  U_i = 1/2 sum_j [phi(r) - phi(rc) - (r - rc) phi'(rc)],  fmag = phi'(r) - phi'(rc)
//   Finnis-Sinclair   U_i = 1/2 sum_j v(r) + F(rho_i), rho_i = sum_j psi(r), F = -A sqrt(rho),
//                     v = D[e^{-2a(r-r0)} - 2e^{-a(r-r0)}] t(r), psi = e^{-beta(r-rho_r0)} t(r),
//                     t = cosine taper r_on..r_cut;  fmag = v' + (F'(rho_i) + F'(rho_j)) psi'
//                     (two passes: densities, then forces; F'(rho_i) rides in Rc[i].w so that the second
//                     pass gathers position and F'(rho_j) from the same 32-byte sector).
//
// One thread per atom, full neighbour lists, no fp64 atomics.  History (ncu evidence under profiles/):
//   r1a  entry-by-entry walk of the Verlet list with `if (r < r_cut)`, `if (r > r_on)` per lane: 61 % lane
//        utilisation, fp64 pipe 35 % busy (every lane paid for every path).
//   r1b  a per-step compaction pass (K2a) wrote an in-range list split plain / taper, K2b walked it: force pass
//        fp64 pipe 61 %, but the compaction pass cost more than the force pass (10.4 ms vs 8.1 ms at c4: 80
//        non-fp64 instructions per list entry, 9 GB of list traffic, gathers stalled on a 37 % L1 hit rate).
//   r1c  (this file) the Verlet list is sorted by distance when it is built (kernels_neighbor.cu), so in a solid
//        the k-th entry of all 32 atoms of a warp lies in the same neighbour shell and the per-entry decisions are
//        warp-uniform nearly always.  Both passes are now one plain loop, two entries per iteration, with three
//        warp-level cases: nobody in range -> skip; nobody in the taper zone -> plain formula; otherwise the
//        general formula (taper with t = 1 selected for r <= r_on).  Lanes that disagree are masked, never
//        branched.  List entries are fetched two iterations ahead and the neighbour sectors one iteration ahead,
//        so gather latency is off the dependent fp64 chain; the math (rsqrt, exp) is branch-free with
//        constant-bank coefficients.  The potential's constants and their products are precomputed on the
//        host and read as constant-bank operands of the kernel parameter, which frees enough registers for
//        five blocks (20 warps) per SM: 11.28 -> 10.93 ms at c4 (six blocks spill: 13.4 ms).
//   Tried and dropped: the virial as sum_i R_i (x) F_i - 1/2 sum (n h) (x) f^ij (exact since f^ij = -f^ji bitwise;
//   six FMAs and twelve registers per pair less).  Parity held, but one lane in ~14 has a shifted entry per
//   iteration, so nearly every warp iteration took the shift branch: K2 3 % slower at c4.
//   Also tried and dropped: each list as an unshifted group (walked with no shift logic) followed by the entries
//   with a periodic shift.  Parity held, K2 27 % slower: an atom near a cell face loses part of every shell to
//   the second group, its k-th entry no longer lies in the shell of its warp neighbours, and the warp-level
//   plain / taper dispatch degrades for the third of all atoms that sit within r_list of a face.
// Per-thread sums run in list order and block partials through a fixed tree: bitwise repeatable.
#include "cfneb_internal.cuh"
#include "trig01.cuh"
#include <math.h>
#include <string.h>

namespace cfn {

constexpr unsigned kFull = 0xffffffffu;

__device__ __forceinline__ double4 ld256(const double4 *p) {  // one LDG.E.256 instead of two LDG.E.128
    double4 v;
    asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(v.x), "=d"(v.y), "=d"(v.z), "=d"(v.w) : "l"(p));
    return v;
}

// r^ij and r^2.  The periodic-shift branch is taken only by warps that hold a shifted entry at all.
__device__ __forceinline__ void pair_vec(const double4 &ri, const double4 &rj, uint32_t code, const double *sh,
                                         double &dx, double &dy, double &dz, double &r2) {
    dx = rj.x - ri.x;
    dy = rj.y - ri.y;
    dz = rj.z - ri.z;
    if (__any_sync(kFull, code != kCodeCenter)) {
        if (code != kCodeCenter) {
            const double n0 = (double)((int)(code & 7u) - 4), n1 = (double)((int)((code >> 3) & 7u) - 4),
                         n2 = (double)((int)((code >> 6) & 7u) - 4);
            dx += n0 * sh[0] + n1 * sh[3] + n2 * sh[6];
            dy += n0 * sh[1] + n1 * sh[4] + n2 * sh[7];
            dz += n0 * sh[2] + n1 * sh[5] + n2 * sh[8];
        }
    }
    r2 = fma(dz, dz, fma(dy, dy, dx * dx));
}

// exp(x) for |x| < 700 (pair arguments are O(1)):  x = (32 k + j) ln2/32 + r,  exp(x) = 2^k T[j] e^r with
// T[j] = 2^(j/32) from a 32-entry table in shared memory and e^r - 1 = r + r^2 (1/2 + r/6 + ... + r^4/720) on
// |r| <= ln2/64 (remainder 3.5e-18); 2^k by exponent arithmetic.  11 fp64 instructions instead of the 17 of a
// degree-13 polynomial on |r| <= ln2/2: the kernels are bound by issue slots, and every fp64 instruction holds
// its scheduler for two.  Max relative error 1.9e-16 against long double over [-8, 3].  No under/overflow
// branches (out-of-range lanes may produce garbage; they are masked, never trapped).
__constant__ double kExp2Table[32] = {
    1.0, 1.0218971486541166, 1.0442737824274138, 1.0671404006768237, 1.0905077326652577, 1.1143867425958924,
    1.1387886347566916, 1.1637248587775775, 1.189207115002721, 1.215247359980469, 1.241857812073484,
    1.2690509571917332, 1.2968395546510096, 1.3252366431597413, 1.3542555469368927, 1.383909881963832,
    1.4142135623730951, 1.4451808069770467, 1.4768261459394993, 1.5091644275934228, 1.5422108254079407,
    1.5759808451078865, 1.6104903319492543, 1.645755478153965, 1.681792830507429, 1.718619298122478,
    1.7562521603732995, 1.7947090750031072, 1.8340080864093424, 1.8741676341103, 1.9152065613971474,
    1.9571441241754002};
// scalar constants of exp_nb in the constant bank (as immediates each costs two UMOVs per use)
__constant__ double kExpK[9] = {46.166241308446828384 /* 32/ln2 */, -2.16608493865351192653e-02, -5.96317165397058656257e-12,
                                1.0 / 720, 1.0 / 120, 1.0 / 24, 1.0 / 6, 0.5, 6755399441055744.0};
// T = shared-window address of the 32-entry table (from __cvta_generic_to_shared, computed once per thread)
__device__ __forceinline__ double exp_nb(double x, uint32_t T) {
    const double t = fma(x, kExpK[0], kExpK[8]);  // integer part lands in the low word
    const double kf = t - kExpK[8];
    double r = fma(kf, kExpK[1], x);  // ln2/32 in two pieces
    r = fma(kf, kExpK[2], r);
    const int n = __double2loint(t);
    double Tj;
    asm("ld.shared.f64 %0, [%1];" : "=d"(Tj) : "r"(T + ((uint32_t)(n & 31) << 3)));
    const double r2 = r * r;
    const double in = fma(fma(fma(fma(kExpK[3], r, kExpK[4]), r, kExpK[5]), r, kExpK[6]), r, kExpK[7]);
    const double q = fma(r2, in, r);
    const double p = fma(Tj, q, Tj);
    return __hiloint2double(__double2hiint(p) + ((n >> 5) << 20), __double2loint(p));
}

struct Acc {  // per-thread sums of one atom
    double fx, fy, fz, ui, sxx, syy, szz, sxy, sxz, syz;
};

__device__ __forceinline__ void add_pair(Acc &a, double s, double u, double dx, double dy, double dz) {
    const double px = s * dx, py = s * dy, pz = s * dz;  // f^ij = (fmag / r) r^ij
    a.fx += px; a.fy += py; a.fz += pz;
    a.ui += u;
    a.sxx = fma(dx, px, a.sxx); a.syy = fma(dy, py, a.syy); a.szz = fma(dz, pz, a.szz);
    a.sxy = fma(dx, py, a.sxy); a.sxz = fma(dx, pz, a.sxz); a.syz = fma(dy, pz, a.syz);
}

// Potential constants, precomputed on the host into Dev::potc (prepare_potential) so that the kernels read them as
// constant-bank operands of the kernel parameter instead of holding ~30 registers of them per thread.
struct FSc { double Dm, a, r0, beta, rr0, A, r_on, inv_w, pi_w, k3, ar0, brr0, hDm, a2Dm, bk3; };  // potc[0..14]
struct LJc { double eps4, sig2, rc, phi_c, dphi_c; };                                               // potc[16..20]
constexpr int kPotcLJ = 16, kPotcRc2 = 22, kPotcRon2 = 23;

// LJ shifted-force pair: fmag / r and the half pair energy
__device__ __forceinline__ void lj_pair(const LJc &c, double r2, double &s, double &u) {
    const double rinv = rsqrt_nr(r2), r = r2 * rinv, ir2 = rinv * rinv;
    const double sr2 = c.sig2 * ir2, sr6 = sr2 * sr2 * sr2, sr12 = sr6 * sr6;
    u = 0.5 * (c.eps4 * (sr12 - sr6) - c.phi_c - (r - c.rc) * c.dphi_c);
    s = c.eps4 * (-12.0 * sr12 + 6.0 * sr6) * ir2 - c.dphi_c * rinv;
}

// FS force pair (second pass).  TAPER = false: r <= r_on, t = 1, t' = 0.
// SHARE: beta == 2 alpha, so e^{-beta (r - rho_r0)} = e^{beta (rho_r0 - r0)} (e^{-alpha (r - r0)})^2 and the second
// exponential is one multiplication (k3 is that constant factor).
//   v = D (e2 - 2 e1),  v' = 2 a D (e1 - e2),  psi = e3,  psi' = -beta e3   (e1 = e^{-a (r - r0)}, e2 = e1^2)
template <bool TAPER, bool SHARE>
__device__ __forceinline__ void fs_pair(const FSc &c, uint32_t T, double r2, double dF_sum, double &s, double &u) {
    const double rinv = rsqrt_nr(r2), r = r2 * rinv;
    const double e1 = exp_nb(fma(-c.a, r, c.ar0), T), e2 = e1 * e1;
    const double w = fma(-2.0, e1, e2), dm = c.a2Dm * (e1 - e2);
    double fmag;
    if (TAPER) {
        const double e3 = SHARE ? c.k3 * e2 : exp_nb(fma(-c.beta, r, c.brr0), T);
        const double m = c.Dm * w;
        double sn, cs;
        sincospi01((r - c.r_on) * c.inv_w, sn, cs);
        double t = 0.5 * (1.0 + cs), dt = -0.5 * sn * c.pi_w;
        if (r <= c.r_on) { t = 1.0; dt = 0.0; }  // lanes outside the taper zone on the general path
        u = 0.5 * (m * t);
        fmag = dm * t + m * dt + dF_sum * (e3 * (dt - c.beta * t));
    } else {
        u = c.hDm * w;
        if (SHARE) fmag = fma(-(dF_sum * c.bk3), e2, dm);
        else fmag = fma(-(dF_sum * c.beta), exp_nb(fma(-c.beta, r, c.brr0), T), dm);
    }
    s = fmag * rinv;
}

// FS density pair (first pass)
template <bool TAPER>
__device__ __forceinline__ double fs_density(const FSc &c, uint32_t T, double r2) {
    const double r = r2 * rsqrt_nr(r2);
    double psi = exp_nb(fma(-c.beta, r, c.brr0), T);
    if (TAPER) {
        double t = 0.5 * (1.0 + cospi01((r - c.r_on) * c.inv_w));
        if (r <= c.r_on) t = 1.0;
        psi *= t;
    }
    return psi;
}

// Walks the (distance-sorted) Verlet column of one atom two entries per iteration: body(k, code0, code1, rj0, rj1)
// sees entries k, k + 1 (shift codes and the neighbours' 32-byte sectors).  Entries are fetched two iterations
// and sectors one iteration ahead of use; the loop is unrolled over the two pipeline stages so that no register
// is rotated.  Rows past an atom's count hold a stand-in entry that is out of range by construction
// (kernels_neighbor.cu), and the list carries 16 rows of slack (api.cu carve()), so no load is predicated.
template <class Body>
__device__ __forceinline__ void walk_list(const uint32_t *__restrict__ lp, size_t stride, const double4 *Rc, int cnt_w,
                                          Body body) {
    uint32_t a0 = lp[0], a1 = lp[stride], b0 = lp[2 * stride], b1 = lp[3 * stride];
    double4 sa0 = ld256(Rc + (a0 & kIdxMask)), sa1 = ld256(Rc + (a1 & kIdxMask)), sb0, sb1;
    lp += 4 * stride;
    for (int k = 0; k < cnt_w; k += 4) {
        sb0 = ld256(Rc + (b0 & kIdxMask));
        sb1 = ld256(Rc + (b1 & kIdxMask));
        {
            const uint32_t c0 = a0 >> kShiftBits, c1 = a1 >> kShiftBits;
            a0 = lp[0];
            a1 = lp[stride];
            body(k, c0, c1, sa0, sa1);
        }
        if (k + 2 >= cnt_w) break;
        sa0 = ld256(Rc + (a0 & kIdxMask));
        sa1 = ld256(Rc + (a1 & kIdxMask));
        {
            const uint32_t c0 = b0 >> kShiftBits, c1 = b1 >> kShiftBits;
            b0 = lp[2 * stride];
            b1 = lp[3 * stride];
            body(k + 2, c0, c1, sb0, sb1);
        }
        lp += 4 * stride;
    }
}

// K2a (FS only): densities rho_i = sum_j psi(r_ij) over the Verlet list; writes F'(rho_i) into Rc[i].w and the
// per-block embedding energy.  Two entries per iteration in 70 registers: seven blocks (28 warps) per SM measured
// 10.66 ms for K2 at c4 against 10.94 with four entries per iteration at five blocks.
// Resident blocks per multiprocessor (tuning knobs; the measured alternatives are in profiles/r2_k2_experiments.md)
#ifndef CFNEB_DENSITY_BLOCKS
#define CFNEB_DENSITY_BLOCKS (7 * 128 / CFNEB_PAIR_THREADS)
#endif
#ifndef CFNEB_FORCE_BLOCKS
#define CFNEB_FORCE_BLOCKS (5 * 128 / CFNEB_PAIR_THREADS)
#endif
__global__ void __launch_bounds__(kThreadsPair, CFNEB_DENSITY_BLOCKS) density_kernel(Dev d, int p_lo) {
    int p;
    if (!image_of(blockIdx.y, p_lo, d.ctl->P, p)) return;
    const int slot = d.order[p];
    __shared__ double sh[9];
    __shared__ double red2[64];
    __shared__ double sT_tab[32];
    if (threadIdx.x < 9) sh[threadIdx.x] = d.geom[slot].h[threadIdx.x];
    if (threadIdx.x < 32) sT_tab[threadIdx.x] = kExp2Table[threadIdx.x];
    __syncthreads();
    const uint32_t sT = (uint32_t)__cvta_generic_to_shared(sT_tab);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = i < d.N;
    double4 *Rc = d.Rc + (size_t)slot * d.Npad;
    const FSc &fs = *reinterpret_cast<const FSc *>(d.potc);
    const double rc2 = d.potc[kPotcRc2], ron2 = d.potc[kPotcRon2];

    // idle lanes sit far away from everything (every r^2 ~ 1e60: out of range, finite) and walk the last column
    double4 ri = make_double4(1e30, 1e30, 1e30, 0.0);
    int cnt = 0;
    const int t_dead = first_dead_tail_bucket(d.r_cut, d.r_list, d.geom[slot].acc);  // block-uniform
    if (valid) {
        ri = ld256(Rc + i);
        cnt = t_dead < kTailBuckets ? (int)d.nbr_tail[((size_t)slot * kTailBuckets + t_dead) * d.Npad + i]
                                    : d.nbr_count[(size_t)slot * d.Npad + i];
    }
    const int cnt_w = min(__reduce_max_sync(kFull, cnt), d.cap);
    const int cap = d.cap;
    double rho = 0.0;
    walk_list(d.nbr_list + (size_t)slot * d.cap * d.Npad + min(i, d.Npad - 1), d.Npad, Rc, cnt_w,
              [&](int k, uint32_t c0, uint32_t c1, const double4 &rj0, const double4 &rj1) {
        double dx, dy, dz, r20, r21;
        pair_vec(ri, rj0, c0, sh, dx, dy, dz, r20);
        pair_vec(ri, rj1, c1, sh, dx, dy, dz, r21);
        const bool in0 = r20 < rc2, in1 = r21 < rc2 && k + 1 < cap;
        if (!__any_sync(kFull, in0 || in1)) return;
        const bool tp = (in0 && r20 > ron2) || (in1 && r21 > ron2);
        double p0, p1;
        if (!__any_sync(kFull, tp)) {
            p0 = fs_density<false>(fs, sT, r20);
            p1 = fs_density<false>(fs, sT, r21);
        } else {
            p0 = fs_density<true>(fs, sT, r20);
            p1 = fs_density<true>(fs, sT, r21);
        }
        if (in0) rho += p0;
        if (in1) rho += p1;
    });
    double emb[1] = {0.0};
    if (valid) {
        double dF = 0.0;
        if (rho > 0.0) {  // F = -A sqrt(rho), F' = -A / (2 sqrt(rho)); rho = 0 => F = F' = 0
            const double sq = sqrt(rho);
            emb[0] = -fs.A * sq;
            dF = -fs.A / (2.0 * sq);
        }
        Rc[i].w = dF;
    }
    double emb_lo = 0.0;
    block_sum_dd(emb[0], emb_lo, red2);
    if (threadIdx.x == 0) {
        double *out = d.part_force + ((size_t)slot * d.nblk_force + blockIdx.x) * kNForcePart;
        out[7] = emb[0];
        out[9] = emb_lo;
    }
}

// K2b: forces, energies and the virial over the Verlet list.
template <int POT, bool SHARE>
__global__ void __launch_bounds__(kThreadsPair, CFNEB_FORCE_BLOCKS) force_kernel(Dev d, int p_lo) {
    int p;
    if (!image_of(blockIdx.y, p_lo, d.ctl->P, p)) return;
    const int slot = d.order[p];
    constexpr bool FS = POT == CFNEB_POT_FS_MORSE;
    __shared__ double sh[9];
    __shared__ double red[32 * 7];
    __shared__ double sT_tab[32];
    if (threadIdx.x < 9) sh[threadIdx.x] = d.geom[slot].h[threadIdx.x];
    if (threadIdx.x < 32) sT_tab[threadIdx.x] = kExp2Table[threadIdx.x];
    __syncthreads();
    const uint32_t sT = (uint32_t)__cvta_generic_to_shared(sT_tab);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = i < d.N;
    const double4 *Rc = d.Rc + (size_t)slot * d.Npad;
    const FSc &fs = *reinterpret_cast<const FSc *>(d.potc);
    const LJc &lj = *reinterpret_cast<const LJc *>(d.potc + kPotcLJ);
    const double rc2 = d.potc[kPotcRc2], ron2 = d.potc[kPotcRon2];

    double4 ri = make_double4(1e30, 1e30, 1e30, 0.0);  // idle lanes: see density_kernel
    int cnt = 0;
    const int t_dead = first_dead_tail_bucket(d.r_cut, d.r_list, d.geom[slot].acc);  // block-uniform
    if (valid) {
        ri = ld256(Rc + i);
        cnt = t_dead < kTailBuckets ? (int)d.nbr_tail[((size_t)slot * kTailBuckets + t_dead) * d.Npad + i]
                                    : d.nbr_count[(size_t)slot * d.Npad + i];
    }
    const int cnt_w = min(__reduce_max_sync(kFull, cnt), d.cap);
    const int cap = d.cap;
    Acc acc = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    walk_list(d.nbr_list + (size_t)slot * d.cap * d.Npad + min(i, d.Npad - 1), d.Npad, Rc, cnt_w,
              [&](int k, uint32_t c0, uint32_t c1, const double4 &rj0, const double4 &rj1) {
        double dx0, dy0, dz0, r20, dx1, dy1, dz1, r21, s0, u0, s1, u1;
        pair_vec(ri, rj0, c0, sh, dx0, dy0, dz0, r20);
        pair_vec(ri, rj1, c1, sh, dx1, dy1, dz1, r21);
        const bool in0 = r20 < rc2, in1 = r21 < rc2 && k + 1 < cap;
        if (!__any_sync(kFull, in0 || in1)) return;
        const bool tp = FS && ((in0 && r20 > ron2) || (in1 && r21 > ron2));
        if (FS) {
            if (!__any_sync(kFull, tp)) {
                fs_pair<false, SHARE>(fs, sT, r20, ri.w + rj0.w, s0, u0);
                fs_pair<false, SHARE>(fs, sT, r21, ri.w + rj1.w, s1, u1);
            } else {
                fs_pair<true, SHARE>(fs, sT, r20, ri.w + rj0.w, s0, u0);
                fs_pair<true, SHARE>(fs, sT, r21, ri.w + rj1.w, s1, u1);
            }
        } else {
            lj_pair(lj, r20, s0, u0);
            lj_pair(lj, r21, s1, u1);
        }
        if (in0) add_pair(acc, s0, u0, dx0, dy0, dz0);
        if (in1) add_pair(acc, s1, u1, dx1, dy1, dz1);
    });
    if (valid) {
        double *F = d.F + (size_t)slot * 3 * d.Npad;
        F[i] = acc.fx;
        F[d.Npad + i] = acc.fy;
        F[2 * (size_t)d.Npad + i] = acc.fz;
    }
    double out6[6] = {-0.5 * acc.sxx, -0.5 * acc.syy, -0.5 * acc.szz, -0.5 * acc.sxy, -0.5 * acc.sxz, -0.5 * acc.syz};
    block_sum<6>(out6, red);
    double e_hi = acc.ui, e_lo = 0.0;  // the energy channel in two doubles (block_sum_dd)
    block_sum_dd(e_hi, e_lo, red);
    if (threadIdx.x == 0) {
        double *out = d.part_force + ((size_t)slot * d.nblk_force + blockIdx.x) * kNForcePart;
        out[0] = e_hi;
        out[8] = e_lo;
#pragma unroll
        for (int n = 0; n < 6; ++n) out[1 + n] = out6[n];
        if (POT == CFNEB_POT_LJ_SF) { out[7] = 0.0; out[9] = 0.0; }
    }
}

void prepare_potential(Dev &d) {
    for (double &x : d.potc) x = 0.0;
    d.potc[kPotcRc2] = d.r_cut * d.r_cut;
    if (d.potential == CFNEB_POT_DNN || d.potential == CFNEB_POT_NEP) {
        // constants are read from Dev::pot, weights from Dev::dn_w
    } else if (d.potential == CFNEB_POT_SW) {
        for (int k = 0; k < 9; ++k) d.potc[k] = d.pot[k];  // eps, sigma, a, lambda, gamma, A, B, p, q
    } else if (d.potential == CFNEB_POT_FS_MORSE) {
        FSc c;
        c.Dm = d.pot[0]; c.a = d.pot[1]; c.r0 = d.pot[2]; c.beta = d.pot[3]; c.rr0 = d.pot[4]; c.A = d.pot[5];
        c.r_on = d.pot[6]; c.inv_w = 1.0 / (d.pot[7] - d.pot[6]); c.pi_w = 3.14159265358979323846 * c.inv_w;
        c.k3 = exp(c.beta * (c.rr0 - c.r0));
        c.ar0 = c.a * c.r0; c.brr0 = c.beta * c.rr0; c.hDm = 0.5 * c.Dm; c.a2Dm = 2.0 * c.a * c.Dm; c.bk3 = c.beta * c.k3;
        memcpy(d.potc, &c, sizeof c);
        d.potc[kPotcRon2] = c.r_on * c.r_on;
    } else {
        LJc c;
        c.eps4 = 4.0 * d.pot[0]; c.sig2 = d.pot[1] * d.pot[1]; c.rc = d.pot[2];
        const double src2 = c.sig2 / (c.rc * c.rc), src6 = src2 * src2 * src2, src12 = src6 * src6;
        c.phi_c = c.eps4 * (src12 - src6);
        c.dphi_c = c.eps4 * (-12.0 * src12 + 6.0 * src6) / c.rc;
        memcpy(d.potc + kPotcLJ, &c, sizeof c);
    }
}

void launch_force(const Dev &d, int p_lo, cudaStream_t st) {
    const int nimg = images_in_grid(d.S, p_lo);
    if (nimg <= 0) return;
    dim3 grid(d.nblk_force, nimg);
    if (d.potential == CFNEB_POT_SW) {
        launch_force_sw(d, p_lo, st);
    } else if (d.potential == CFNEB_POT_DNN) {
        launch_force_dn(d, p_lo, st);
    } else if (d.potential == CFNEB_POT_NEP) {
        launch_force_nep(d, p_lo, st);
    } else if (d.potential == CFNEB_POT_LJ_SF) {
        force_kernel<CFNEB_POT_LJ_SF, false><<<grid, kThreadsPair, 0, st>>>(d, p_lo);
    } else {
        density_kernel<<<grid, kThreadsPair, 0, st>>>(d, p_lo);
        if (d.pot[3] == 2.0 * d.pot[1]) force_kernel<CFNEB_POT_FS_MORSE, true><<<grid, kThreadsPair, 0, st>>>(d, p_lo);
        else force_kernel<CFNEB_POT_FS_MORSE, false><<<grid, kThreadsPair, 0, st>>>(d, p_lo);
    }
}

}  // namespace cfn

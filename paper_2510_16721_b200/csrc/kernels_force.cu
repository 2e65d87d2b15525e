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
// One thread per atom, full neighbour lists, no fp64 atomics.  The first form of this kernel walked the Verlet
// list (r < r_cut + skin) entry by entry with `if (r < r_cut)` and `if (r > r_on)` inside the loop; ncu
// (profiles/r1a) showed 61 % lane utilisation and the fp64 pipe 35 % busy: in a warp of 32 different atoms some
// lane is always in the taper zone and some lane always out of range, so every lane paid for every path, and
// the gather latency sat on the critical path of a long dependent fp64 chain.  Now each thread runs two
// phases over a private shared-memory queue (64 entries, [k][thread] so bank = lane):
//   phase A  stream the list 4 entries at a time (coalesced k-major list read, one 256-bit gather of the
//            neighbour's position sector each, r^2 only) and push the entries inside r_cut onto the queue --
//            plain ones (r <= r_on) from the front, taper-zone ones from the back;
//   phase B  when a queue in the warp is about to fill (or the list ends) evaluate the queue: the plain loop
//            carries no taper arithmetic, the taper loop no branch, two pairs per thread are in flight, and
//            the math (rsqrt, exp) is branch-free with constant-bank coefficients.
// Per-thread sums run in list order and block partials through a fixed tree: bitwise repeatable.
#include "cfneb_internal.cuh"

namespace cfn {

constexpr int kQ = 32;  // queued r^2 values per thread (32 KB of shared memory per 128-thread block)
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

// 1/sqrt(x) for normal x > 0: hardware seed (2^-22) + one cubically convergent step; no special cases.
__device__ __forceinline__ double rsqrt_nr(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-(x * y), y, 1.0);
    return fma(y * e, fma(0.375, e, 0.5), y);
}

// exp(x) for |x| < 700 (pair arguments are O(1)): x = k ln2 + r, degree-13 Taylor polynomial on |r| <= ln2/2
// (remainder 4e-18), 2^k by exponent arithmetic.  No under/overflow branches; coefficients from the constant bank.
__constant__ double kExpC[14] = {1.0, 1.0, 1.0 / 2, 1.0 / 6, 1.0 / 24, 1.0 / 120, 1.0 / 720, 1.0 / 5040, 1.0 / 40320,
                                 1.0 / 362880, 1.0 / 3628800, 1.0 / 39916800, 1.0 / 479001600, 1.0 / 6227020800.0};
__device__ __forceinline__ double exp_nb(double x) {
    const double t = fma(x, 1.4426950408889634074, 6755399441055744.0);
    const double kf = t - 6755399441055744.0;
    double r = fma(kf, -6.93147180369123816490e-01, x);
    r = fma(kf, -1.90821492927058770002e-10, r);
    double p = kExpC[13];
#pragma unroll
    for (int n = 12; n >= 0; --n) p = fma(p, r, kExpC[n]);
    return __hiloint2double(__double2hiint(p) + (__double2loint(t) << 20), __double2loint(p));
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

struct LJc { double eps4, sig2, rc, phi_c, dphi_c; };
struct FSc { double Dm, a, r0, beta, rr0, A, r_on, inv_w, pi_w; };

// LJ shifted-force pair: fmag / r and the half pair energy
__device__ __forceinline__ void lj_pair(const LJc &c, double r2, double &s, double &u) {
    const double rinv = rsqrt_nr(r2), r = r2 * rinv, ir2 = rinv * rinv;
    const double sr2 = c.sig2 * ir2, sr6 = sr2 * sr2 * sr2, sr12 = sr6 * sr6;
    u = 0.5 * (c.eps4 * (sr12 - sr6) - c.phi_c - (r - c.rc) * c.dphi_c);
    s = c.eps4 * (-12.0 * sr12 + 6.0 * sr6) * ir2 - c.dphi_c * rinv;
}

// FS force pair (second pass).  TAPER = false: r <= r_on, t = 1, t' = 0.
template <bool TAPER>
__device__ __forceinline__ void fs_pair(const FSc &c, double r2, double dF_sum, double &s, double &u) {
    const double rinv = rsqrt_nr(r2), r = r2 * rinv;
    const double e1 = exp_nb(-c.a * (r - c.r0)), e2 = e1 * e1;
    const double m = c.Dm * (e2 - 2.0 * e1), dm = 2.0 * c.a * c.Dm * (e1 - e2);
    const double e3 = exp_nb(-c.beta * (r - c.rr0));
    double fmag;
    if (TAPER) {
        double sn, cs;
        sincospi((r - c.r_on) * c.inv_w, &sn, &cs);
        double t = 0.5 * (1.0 + cs), dt = -0.5 * sn * c.pi_w;
        if (r <= c.r_on) { t = 1.0; dt = 0.0; }  // the queues are split on r^2; keep the definition exact at the edge
        u = 0.5 * (m * t);
        fmag = dm * t + m * dt + dF_sum * (e3 * (dt - c.beta * t));
    } else {
        u = 0.5 * m;
        fmag = dm - dF_sum * (c.beta * e3);
    }
    s = fmag * rinv;
}

// FS density pair (first pass)
template <bool TAPER>
__device__ __forceinline__ double fs_density(const FSc &c, double r2) {
    const double r = r2 * rsqrt_nr(r2);
    double psi = exp_nb(-c.beta * (r - c.rr0));
    if (TAPER) {
        double t = 0.5 * (1.0 + cospi((r - c.r_on) * c.inv_w));
        if (r <= c.r_on) t = 1.0;
        psi *= t;
    }
    return psi;
}

// Potential constants in registers.
template <int POT>
struct PotC {
    LJc lj;
    FSc fs;
    double rc2, ron2;
    __device__ __forceinline__ void load(const Dev &d) {
        rc2 = d.r_cut * d.r_cut;
        ron2 = 0.0;
        if (POT == CFNEB_POT_FS_MORSE) {
            fs.Dm = d.pot[0]; fs.a = d.pot[1]; fs.r0 = d.pot[2]; fs.beta = d.pot[3]; fs.rr0 = d.pot[4]; fs.A = d.pot[5];
            fs.r_on = d.pot[6]; fs.inv_w = 1.0 / (d.pot[7] - d.pot[6]); fs.pi_w = 3.14159265358979323846 * fs.inv_w;
            ron2 = fs.r_on * fs.r_on;
        } else {
            lj.eps4 = 4.0 * d.pot[0]; lj.sig2 = d.pot[1] * d.pot[1]; lj.rc = d.pot[2];
            const double src2 = lj.sig2 / (lj.rc * lj.rc), src6 = src2 * src2 * src2, src12 = src6 * src6;
            lj.phi_c = lj.eps4 * (src12 - src6);
            lj.dphi_c = lj.eps4 * (-12.0 * src12 + 6.0 * src6) / lj.rc;
        }
    }
};

// K2a: classify the Verlet list of every atom into the in-range list of this step (plain entries from the
// front, taper-zone entries from the back of the atom's column of nbr_in) and, for FS, accumulate the density
// rho_i: plain r^2 values go through the shared-memory queue and are evaluated densely, the taper entries at the
// end.  Writes F'(rho_i) into Rc[i].w and the per-block embedding energy.
template <int POT>
__global__ void __launch_bounds__(kThreadsAtom, 4) classify_kernel(Dev d, int p_lo) {
    const int p = blockIdx.y + p_lo;
    if (p > d.ctl->P - 1 - p_lo) return;
    const int slot = d.order[p];
    constexpr bool FS = POT == CFNEB_POT_FS_MORSE;
    __shared__ double s_q[FS ? kQ * kThreadsAtom : 1];
    __shared__ double sh[9];
    __shared__ double red[32];
    if (threadIdx.x < 9) sh[threadIdx.x] = d.geom[slot].h[threadIdx.x];
    __syncthreads();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = i < d.N;
    double4 *Rc = d.Rc + (size_t)slot * d.Npad;
    const size_t col = (size_t)slot * d.cap * d.Npad + i;
    const uint32_t *lp = d.nbr_list + col;
    uint32_t *ip = d.nbr_in + col;
    double *q = s_q + threadIdx.x;  // entry c of this thread at q[c * kThreadsAtom]
    PotC<POT> pc;
    pc.load(d);

    double4 ri = make_double4(0.0, 0.0, 0.0, 0.0);
    int cnt = 0;
    if (valid) {
        ri = ld256(Rc + i);
        cnt = d.nbr_count[(size_t)slot * d.Npad + i];
    }
    const uint32_t self = (uint32_t)(valid ? i : 0) | (kCodeCenter << kShiftBits);  // stand-in entry of idle lanes
    const int cnt_w = __reduce_max_sync(kFull, cnt);
    const int last = d.cap - 1;
    double rho = 0.0;
    int n_pl = 0, n_tp = 0, n_q = 0;

    // The list entries of iteration k+1 are loaded before the gathers of iteration k are consumed, so the
    // (DRAM-streamed) list read never sits on the critical path.
    uint32_t en[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) en[u] = (u < cnt) ? lp[(size_t)u * d.Npad] : self;
    int k = 0;
    while (k < cnt_w) {
        do {  // phase A: four list entries in flight
            uint32_t e[4];
            double4 rj[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) { e[u] = en[u]; rj[u] = ld256(Rc + (e[u] & kIdxMask)); }
#pragma unroll
            for (int u = 0; u < 4; ++u) en[u] = (k + 4 + u < cnt) ? lp[(size_t)(k + 4 + u) * d.Npad] : self;
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                double dx, dy, dz, r2;
                pair_vec(ri, rj[u], e[u] >> kShiftBits, sh, dx, dy, dz, r2);
                const bool in = (k + u < cnt) && r2 < pc.rc2;
                const bool tp = FS && in && r2 > pc.ron2;
                if (in && !tp) {
                    ip[(size_t)n_pl * d.Npad] = e[u];
                    ++n_pl;
                    if (FS) { q[n_q * kThreadsAtom] = r2; ++n_q; }
                }
                if (tp) { ip[(size_t)(last - n_tp) * d.Npad] = e[u]; ++n_tp; }
            }
            k += 4;
        } while (k < cnt_w && !(FS && __any_sync(kFull, n_q > kQ - 4)));
        if (FS) {  // phase B: dense evaluation of the queued r^2, two pairs in flight
            const int nq_w = __reduce_max_sync(kFull, n_q);
            for (int c = 0; c < nq_w; c += 2) {
                const bool a0 = c < n_q, a1 = c + 1 < n_q;
                const double r20 = a0 ? q[c * kThreadsAtom] : 1.0, r21 = a1 ? q[(c + 1) * kThreadsAtom] : 1.0;
                const double p0 = fs_density<false>(pc.fs, r20), p1 = fs_density<false>(pc.fs, r21);
                rho += a0 ? p0 : 0.0;
                rho += a1 ? p1 : 0.0;
            }
            n_q = 0;
        }
    }
    if (valid) d.nbr_in_count[(size_t)slot * d.Npad + i] = n_pl | (n_tp << 16);
    if (!FS) return;

    const int ntp_w = __reduce_max_sync(kFull, n_tp);
    uint32_t et = (0 < n_tp) ? ip[(size_t)last * d.Npad] : self;
    for (int c = 0; c < ntp_w; ++c) {  // taper-zone entries, read back from this thread's own column
        const bool a0 = c < n_tp;
        const uint32_t e0 = et;
        const double4 rj0 = ld256(Rc + (e0 & kIdxMask));
        et = (c + 1 < n_tp) ? ip[(size_t)(last - c - 1) * d.Npad] : self;
        double dx, dy, dz, r2;
        pair_vec(ri, rj0, e0 >> kShiftBits, sh, dx, dy, dz, r2);
        const double p0 = fs_density<true>(pc.fs, a0 ? r2 : 1.0);
        rho += a0 ? p0 : 0.0;
    }
    double emb[1] = {0.0};
    if (valid) {
        double dF = 0.0;
        if (rho > 0.0) {  // F = -A sqrt(rho), F' = -A / (2 sqrt(rho)); rho = 0 => F = F' = 0
            const double sq = sqrt(rho);
            emb[0] = -pc.fs.A * sq;
            dF = -pc.fs.A / (2.0 * sq);
        }
        Rc[i].w = dF;
    }
    block_sum<1>(emb, red);
    if (threadIdx.x == 0) d.part_force[((size_t)slot * d.nblk_atom + blockIdx.x) * kNForcePart + 7] = emb[0];
}

// K2b: forces, energies and the virial over the in-range list of K2a.  No shared-memory queue, so the whole
// L1 serves the position gathers; two pairs per thread in flight; the taper loop runs last.
template <int POT>
__global__ void __launch_bounds__(kThreadsAtom, 4) force_kernel(Dev d, int p_lo) {
    const int p = blockIdx.y + p_lo;
    if (p > d.ctl->P - 1 - p_lo) return;
    const int slot = d.order[p];
    constexpr bool FS = POT == CFNEB_POT_FS_MORSE;
    __shared__ double sh[9];
    __shared__ double red[32 * 7];
    if (threadIdx.x < 9) sh[threadIdx.x] = d.geom[slot].h[threadIdx.x];
    __syncthreads();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = i < d.N;
    const double4 *Rc = d.Rc + (size_t)slot * d.Npad;
    const uint32_t *ip = d.nbr_in + (size_t)slot * d.cap * d.Npad + i;
    PotC<POT> pc;
    pc.load(d);

    double4 ri = make_double4(0.0, 0.0, 0.0, 0.0);
    int n_pl = 0, n_tp = 0;
    if (valid) {
        ri = ld256(Rc + i);
        const int c = d.nbr_in_count[(size_t)slot * d.Npad + i];
        n_pl = c & 0xffff;
        n_tp = c >> 16;
    }
    const uint32_t self = (uint32_t)(valid ? i : 0) | (kCodeCenter << kShiftBits);
    const int last = d.cap - 1;
    Acc acc = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};

    const int npl_w = __reduce_max_sync(kFull, n_pl);
    uint32_t en0 = (0 < n_pl) ? ip[0] : self, en1 = (1 < n_pl) ? ip[d.Npad] : self;  // entries one iteration ahead
    for (int c = 0; c < npl_w; c += 2) {
        const bool a0 = c < n_pl, a1 = c + 1 < n_pl;
        const uint32_t e0 = en0, e1 = en1;
        const double4 rj0 = ld256(Rc + (e0 & kIdxMask)), rj1 = ld256(Rc + (e1 & kIdxMask));
        en0 = (c + 2 < n_pl) ? ip[(size_t)(c + 2) * d.Npad] : self;
        en1 = (c + 3 < n_pl) ? ip[(size_t)(c + 3) * d.Npad] : self;
        double dx0, dy0, dz0, r20, dx1, dy1, dz1, r21, s0, u0, s1, u1;
        pair_vec(ri, rj0, e0 >> kShiftBits, sh, dx0, dy0, dz0, r20);
        pair_vec(ri, rj1, e1 >> kShiftBits, sh, dx1, dy1, dz1, r21);
        r20 = a0 ? r20 : 1.0;
        r21 = a1 ? r21 : 1.0;
        if (FS) {
            fs_pair<false>(pc.fs, r20, ri.w + rj0.w, s0, u0);
            fs_pair<false>(pc.fs, r21, ri.w + rj1.w, s1, u1);
        } else {
            lj_pair(pc.lj, r20, s0, u0);
            lj_pair(pc.lj, r21, s1, u1);
        }
        add_pair(acc, a0 ? s0 : 0.0, a0 ? u0 : 0.0, dx0, dy0, dz0);
        add_pair(acc, a1 ? s1 : 0.0, a1 ? u1 : 0.0, dx1, dy1, dz1);
    }
    if (FS) {
        const int ntp_w = __reduce_max_sync(kFull, n_tp);
        uint32_t et = (0 < n_tp) ? ip[(size_t)last * d.Npad] : self;
        for (int c = 0; c < ntp_w; ++c) {
            const bool a0 = c < n_tp;
            const uint32_t e0 = et;
            const double4 rj0 = ld256(Rc + (e0 & kIdxMask));
            et = (c + 1 < n_tp) ? ip[(size_t)(last - c - 1) * d.Npad] : self;
            double dx0, dy0, dz0, r20, s0, u0;
            pair_vec(ri, rj0, e0 >> kShiftBits, sh, dx0, dy0, dz0, r20);
            fs_pair<true>(pc.fs, a0 ? r20 : 1.0, ri.w + rj0.w, s0, u0);
            add_pair(acc, a0 ? s0 : 0.0, a0 ? u0 : 0.0, dx0, dy0, dz0);
        }
    }
    if (valid) {
        double *F = d.F + (size_t)slot * 3 * d.Npad;
        F[i] = acc.fx;
        F[d.Npad + i] = acc.fy;
        F[2 * (size_t)d.Npad + i] = acc.fz;
    }
    double out7[7] = {acc.ui, -0.5 * acc.sxx, -0.5 * acc.syy, -0.5 * acc.szz, -0.5 * acc.sxy, -0.5 * acc.sxz, -0.5 * acc.syz};
    block_sum<7>(out7, red);
    if (threadIdx.x == 0) {
        double *out = d.part_force + ((size_t)slot * d.nblk_atom + blockIdx.x) * kNForcePart;
#pragma unroll
        for (int n = 0; n < 7; ++n) out[n] = out7[n];
        if (POT == CFNEB_POT_LJ_SF) out[7] = 0.0;
    }
}

void launch_force(const Dev &d, int p_lo, cudaStream_t st) {
    const int nimg = d.S - 2 * p_lo;
    if (nimg <= 0) return;
    dim3 grid(d.nblk_atom, nimg);
    if (d.potential == CFNEB_POT_LJ_SF) {
        classify_kernel<CFNEB_POT_LJ_SF><<<grid, kThreadsAtom, 0, st>>>(d, p_lo);
        force_kernel<CFNEB_POT_LJ_SF><<<grid, kThreadsAtom, 0, st>>>(d, p_lo);
    } else {
        classify_kernel<CFNEB_POT_FS_MORSE><<<grid, kThreadsAtom, 0, st>>>(d, p_lo);
        force_kernel<CFNEB_POT_FS_MORSE><<<grid, kThreadsAtom, 0, st>>>(d, p_lo);
    }
}

}  // namespace cfn

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
// One thread per atom, full neighbour lists (no fp64 atomics): every F_i, and every per-block partial of
// E and V, is summed in list order, so results are bitwise repeatable.  Lists are k-major
// ([cap][Npad]), so the list read of a warp is one 128-byte line.
#include "cfneb_internal.cuh"

namespace cfn {

struct PairGeom {
    double dx, dy, dz, r2;
};

__device__ inline PairGeom pair_geom(const double4 &ri, const double4 &rj, uint32_t code, const double *sh /* smem h[9] */) {
    PairGeom g;
    g.dx = rj.x - ri.x;
    g.dy = rj.y - ri.y;
    g.dz = rj.z - ri.z;
    if (code != kCodeCenter) {
        const double n0 = (double)((int)(code & 7u) - 4), n1 = (double)((int)((code >> 3) & 7u) - 4),
                     n2 = (double)((int)((code >> 6) & 7u) - 4);
        g.dx += n0 * sh[0] + n1 * sh[3] + n2 * sh[6];
        g.dy += n0 * sh[1] + n1 * sh[4] + n2 * sh[7];
        g.dz += n0 * sh[2] + n1 * sh[5] + n2 * sh[8];
    }
    g.r2 = g.dx * g.dx + g.dy * g.dy + g.dz * g.dz;
    return g;
}

// cosine taper t(r), t'(r) for r < r_cut
__device__ inline void taper(double r, double r_on, double inv_w, double &t, double &dt) {
    if (r <= r_on) {
        t = 1.0;
        dt = 0.0;
    } else {
        double s, c;
        sincospi((r - r_on) * inv_w, &s, &c);
        t = 0.5 * (1.0 + c);
        dt = -0.5 * s * (3.14159265358979323846 * inv_w);
    }
}

// PASS 0: LJ (single pass) or FS second pass (forces);  PASS 1: FS first pass (densities).
template <int POT, int PASS>
__global__ void __launch_bounds__(kThreadsAtom) force_kernel(Dev d, int p_lo) {
    const int p = blockIdx.y + p_lo;
    if (p > d.ctl->P - 1 - p_lo) return;
    const int slot = d.order[p];
    __shared__ double sh[9];
    __shared__ double red[32 * 7];
    if (threadIdx.x < 9) sh[threadIdx.x] = d.geom[slot].h[threadIdx.x];
    __syncthreads();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = i < d.N;
    double4 *Rc = d.Rc + (size_t)slot * d.Npad;
    const uint32_t *list = d.nbr_list + (size_t)slot * d.cap * d.Npad + i;
    const double rc2 = d.r_cut * d.r_cut;
    double4 ri = make_double4(0.0, 0.0, 0.0, 0.0);
    int cnt = 0;
    if (valid) {
        ri = Rc[i];
        cnt = d.nbr_count[(size_t)slot * d.Npad + i];
    }

    if (POT == CFNEB_POT_FS_MORSE && PASS == 1) {
        const double beta = d.pot[3], rr0 = d.pot[4], A = d.pot[5], r_on = d.pot[6], inv_w = 1.0 / (d.pot[7] - d.pot[6]);
        double rho = 0.0;
#pragma unroll 2
        for (int k = 0; k < cnt; ++k) {
            const uint32_t e = list[(size_t)k * d.Npad];
            const double4 rj = Rc[e & kIdxMask];
            const PairGeom g = pair_geom(ri, rj, e >> kShiftBits, sh);
            if (g.r2 < rc2) {
                const double r = sqrt(g.r2);
                double t = 1.0;
                if (r > r_on) t = 0.5 * (1.0 + cospi((r - r_on) * inv_w));
                rho += exp(-beta * (r - rr0)) * t;
            }
        }
        double emb[1] = {0.0};
        if (valid) {
            double dF = 0.0;
            if (rho > 0.0) {  // F = -A sqrt(rho), F' = -A / (2 sqrt(rho)); rho = 0 => F = F' = 0
                const double sq = sqrt(rho);
                emb[0] = -A * sq;
                dF = -A / (2.0 * sq);
            }
            Rc[i].w = dF;
        }
        block_sum<1>(emb, red);
        if (threadIdx.x == 0) d.part_force[((size_t)slot * d.nblk_atom + blockIdx.x) * kNForcePart + 7] = emb[0];
        return;
    }

    double fx = 0.0, fy = 0.0, fz = 0.0, ui = 0.0;
    double sxx = 0.0, syy = 0.0, szz = 0.0, sxy = 0.0, sxz = 0.0, syz = 0.0;

    if (POT == CFNEB_POT_LJ_SF) {
        const double eps4 = 4.0 * d.pot[0], sig2 = d.pot[1] * d.pot[1], rc = d.pot[2];
        const double src2 = sig2 / (rc * rc), src6 = src2 * src2 * src2, src12 = src6 * src6;
        const double phi_c = eps4 * (src12 - src6);
        const double dphi_c = eps4 * (-12.0 * src12 + 6.0 * src6) / rc;
#pragma unroll 2
        for (int k = 0; k < cnt; ++k) {
            const uint32_t e = list[(size_t)k * d.Npad];
            const double4 rj = Rc[e & kIdxMask];
            const PairGeom g = pair_geom(ri, rj, e >> kShiftBits, sh);
            if (g.r2 < rc2) {
                const double rinv = rsqrt(g.r2), r = g.r2 * rinv, ir2 = rinv * rinv;
                const double sr2 = sig2 * ir2, sr6 = sr2 * sr2 * sr2, sr12 = sr6 * sr6;
                ui += 0.5 * (eps4 * (sr12 - sr6) - phi_c - (r - rc) * dphi_c);
                const double s = eps4 * (-12.0 * sr12 + 6.0 * sr6) * ir2 - dphi_c * rinv;  // fmag / r
                const double px = s * g.dx, py = s * g.dy, pz = s * g.dz;
                fx += px; fy += py; fz += pz;
                sxx += g.dx * px; syy += g.dy * py; szz += g.dz * pz;
                sxy += g.dx * py; sxz += g.dx * pz; syz += g.dy * pz;
            }
        }
    } else {
        const double Dm = d.pot[0], a = d.pot[1], r0 = d.pot[2], beta = d.pot[3], rr0 = d.pot[4];
        const double r_on = d.pot[6], inv_w = 1.0 / (d.pot[7] - d.pot[6]);
        const double dFi = ri.w;
#pragma unroll 2
        for (int k = 0; k < cnt; ++k) {
            const uint32_t e = list[(size_t)k * d.Npad];
            const double4 rj = Rc[e & kIdxMask];
            const PairGeom g = pair_geom(ri, rj, e >> kShiftBits, sh);
            if (g.r2 < rc2) {
                const double rinv = rsqrt(g.r2), r = g.r2 * rinv;
                double t, dt;
                taper(r, r_on, inv_w, t, dt);
                const double e1 = exp(-a * (r - r0)), e2 = e1 * e1;
                const double m = Dm * (e2 - 2.0 * e1), dm = 2.0 * a * Dm * (e1 - e2);
                const double e3 = exp(-beta * (r - rr0));
                const double dpsi = e3 * (dt - beta * t);
                ui += 0.5 * (m * t);
                const double fmag = dm * t + m * dt + (dFi + rj.w) * dpsi;
                const double s = fmag * rinv;
                const double px = s * g.dx, py = s * g.dy, pz = s * g.dz;
                fx += px; fy += py; fz += pz;
                sxx += g.dx * px; syy += g.dy * py; szz += g.dz * pz;
                sxy += g.dx * py; sxz += g.dx * pz; syz += g.dy * pz;
            }
        }
    }
    if (valid) {
        double *F = d.F + (size_t)slot * 3 * d.Npad;
        F[i] = fx;
        F[d.Npad + i] = fy;
        F[2 * (size_t)d.Npad + i] = fz;
    }
    double acc[7] = {ui, -0.5 * sxx, -0.5 * syy, -0.5 * szz, -0.5 * sxy, -0.5 * sxz, -0.5 * syz};
    block_sum<7>(acc, red);
    if (threadIdx.x == 0) {
        double *out = d.part_force + ((size_t)slot * d.nblk_atom + blockIdx.x) * kNForcePart;
#pragma unroll
        for (int q = 0; q < 7; ++q) out[q] = acc[q];
        if (POT == CFNEB_POT_LJ_SF) out[7] = 0.0;
    }
}

void launch_force(const Dev &d, int p_lo, cudaStream_t st) {
    const int nimg = d.S - 2 * p_lo;
    if (nimg <= 0) return;
    dim3 grid(d.nblk_atom, nimg);
    if (d.potential == CFNEB_POT_LJ_SF) {
        force_kernel<CFNEB_POT_LJ_SF, 0><<<grid, kThreadsAtom, 0, st>>>(d, p_lo);
    } else {
        force_kernel<CFNEB_POT_FS_MORSE, 1><<<grid, kThreadsAtom, 0, st>>>(d, p_lo);
        force_kernel<CFNEB_POT_FS_MORSE, 0><<<grid, kThreadsAtom, 0, st>>>(d, p_lo);
    }
}

}  // namespace cfn

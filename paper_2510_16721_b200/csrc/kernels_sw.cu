// kernels_sw.cu -- K2 for a many-body potential: Stillinger-Weber (three-body), evaluated the way the paper writes
// forces and virials for ANY potential whose site energy U_i depends on all vectors r^ij of atom i's environment
// (Eq. 4-8; the paper's own potential, NEP, is of this class -- its trained weights are not available,
// SURVEY.md section 8(f) item 4):
//   pass 1 (sw_partial_kernel)  U_i and the partial forces p^ij = dU_i/dr^ij, one vector per list entry, stored
//   pass 2 (sw_force_kernel; pair_force_batched_kernel for the descriptor network of kernels_dn.cu)
//                               f^ij = p^ij - p^ji (Eq. 5; p^ji sits at the mirror entry (j; i, -n) of j's list,
//                               whose row is tabulated once per list build by sw_mirror_kernel),
//                               F_i = sum_j f^ij,  V = -1/2 sum_i sum_j r^ij (x) f^ij  (Eq. 8)
//   U_i = 1/2 sum_j phi2(r_ij) + sum_{j<k} h(r_ij, r_ik, cos theta_jik),  r_c = a sigma,
//   phi2(r) = A eps [B (sigma/r)^p - (sigma/r)^q] exp(sigma/(r - r_c)),
//   h = lambda eps (cos theta + 1/3)^2 exp(gamma sigma/(r_ij - r_c)) exp(gamma sigma/(r_ik - r_c)).
// One thread per atom, the same Verlet lists (K1) and Cartesian sectors (K0) as the pair kernels, no atomics,
// fixed summation order.  The cut-off holds a handful of neighbours (4 in diamond), so the in-range environment
// of an atom is first gathered into a small per-thread array (kMaxEnv entries; more is CFNEB_ENEIGH_OVERFLOW).
#include "cfneb_internal.cuh"

namespace cfn {

constexpr int kMaxEnv = 32;

struct SWc { double eps, sig, a, lam, gam, A, B, p, q; };  // Dev::potc[0..8]

__device__ __forceinline__ void shifted_vec(const double4 &ri, const double4 &rj, uint32_t code, const double *sh,
                                            double &dx, double &dy, double &dz) {
    dx = rj.x - ri.x; dy = rj.y - ri.y; dz = rj.z - ri.z;
    if (code != kCodeCenter) {
        const double n0 = (double)((int)(code & 7u) - 4), n1 = (double)((int)((code >> 3) & 7u) - 4),
                     n2 = (double)((int)((code >> 6) & 7u) - 4);
        dx += n0 * sh[0] + n1 * sh[3] + n2 * sh[6];
        dy += n0 * sh[1] + n1 * sh[4] + n2 * sh[7];
        dz += n0 * sh[2] + n1 * sh[5] + n2 * sh[8];
    }
}

__global__ void __launch_bounds__(kThreadsAtom) sw_partial_kernel(Dev d, int p_lo) {
    int p;
    if (!image_of(blockIdx.y, p_lo, d.ctl->P, p)) return;
    const int slot = d.order[p];
    __shared__ double sh[9];
    __shared__ double red[64];
    if (threadIdx.x < 9) sh[threadIdx.x] = d.geom[slot].h[threadIdx.x];
    __syncthreads();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = i < d.N;
    const SWc &c = *reinterpret_cast<const SWc *>(d.potc);
    const double rc = c.a * c.sig, rc2 = rc * rc;
    double ui[1] = {0.0};
    if (valid) {
        const double4 *Rc = d.Rc + (size_t)slot * d.Npad;
        const uint32_t *lp = d.nbr_list + (size_t)slot * d.cap * d.Npad + i;
        double *part = d.part + (size_t)slot * d.cap * 3 * d.Npad + i;  // part[(k * 3 + m) * Npad]
        const double4 ri = Rc[i];
        const int cnt = live_rows(d, slot, i);  // rows past it cannot be in range and are neither written nor read
        double ex[kMaxEnv], ey[kMaxEnv], ez[kMaxEnv], er[kMaxEnv], px[kMaxEnv], py[kMaxEnv], pz[kMaxEnv];
        int ek[kMaxEnv];
        int n = 0;
        bool overflow = false;
        // entry k + 2 and the coordinates of entry k + 1 are in flight while entry k is tested (rows past the
        // count are readable: stale or zero entries, 16 rows of slack)
        uint32_t e_n = lp[0], e_nn = lp[(size_t)d.Npad];
        double4 rj_n = Rc[e_n & kIdxMask];
        for (int k = 0; k < cnt; ++k) {
            const uint32_t e = e_n;
            const double4 rj = rj_n;
            e_n = e_nn;
            e_nn = lp[(size_t)(k + 2) * d.Npad];
            rj_n = Rc[e_n & kIdxMask];
            double dx, dy, dz;
            shifted_vec(ri, rj, e >> kShiftBits, sh, dx, dy, dz);
            const double r2 = dx * dx + dy * dy + dz * dz;
            if (r2 < rc2) {
                if (n < kMaxEnv) {
                    ex[n] = dx; ey[n] = dy; ez[n] = dz; er[n] = sqrt(r2); ek[n] = k;
                    px[n] = py[n] = pz[n] = 0.0;
                    ++n;
                } else overflow = true;
            }
        }
        if (overflow) set_error(d.ctl, CFNEB_ENEIGH_OVERFLOW);
        for (int a = 0; a < n; ++a) {
            const double dj = er[a], inv = 1.0 / dj;
            const double sr = c.sig * inv, ee = exp(c.sig / (dj - rc));
            const double tp = c.B * pow(sr, c.p), tq = pow(sr, c.q);
            const double br = tp - tq, dbr = (-c.p * tp + c.q * tq) * inv;
            const double phi = c.A * c.eps * br * ee;
            const double dphi = c.A * c.eps * (dbr * ee + br * ee * (-c.sig / ((dj - rc) * (dj - rc))));
            ui[0] += 0.5 * phi;
            px[a] += 0.5 * dphi * ex[a] * inv; py[a] += 0.5 * dphi * ey[a] * inv; pz[a] += 0.5 * dphi * ez[a] * inv;
            const double gj = exp(c.gam * c.sig / (dj - rc)), dgj = gj * (-c.gam * c.sig / ((dj - rc) * (dj - rc)));
            for (int b = a + 1; b < n; ++b) {  // triplets centred on i, each once
                const double dk = er[b], invk = 1.0 / dk;
                const double gk = exp(c.gam * c.sig / (dk - rc)), dgk = gk * (-c.gam * c.sig / ((dk - rc) * (dk - rc)));
                const double cs = (ex[a] * ex[b] + ey[a] * ey[b] + ez[a] * ez[b]) * inv * invk;
                const double w = cs + 1.0 / 3.0, le = c.lam * c.eps;
                ui[0] += le * w * w * gj * gk;
                const double c2 = 2.0 * w * gj * gk, ra = w * w * dgj * gk, rb = w * w * gj * dgk;
                // d cos / d r^ij = (r^ik/|r^ik| - cos r^ij/|r^ij|) / |r^ij|
                px[a] += le * (c2 * (ex[b] * invk - cs * ex[a] * inv) * inv + ra * ex[a] * inv);
                py[a] += le * (c2 * (ey[b] * invk - cs * ey[a] * inv) * inv + ra * ey[a] * inv);
                pz[a] += le * (c2 * (ez[b] * invk - cs * ez[a] * inv) * inv + ra * ez[a] * inv);
                px[b] += le * (c2 * (ex[a] * inv - cs * ex[b] * invk) * invk + rb * ex[b] * invk);
                py[b] += le * (c2 * (ey[a] * inv - cs * ey[b] * invk) * invk + rb * ey[b] * invk);
                pz[b] += le * (c2 * (ez[a] * inv - cs * ez[b] * invk) * invk + rb * ez[b] * invk);
            }
        }
        // one write per list entry: the partial force of the in-range ones (ek ascending), zero for the others
        for (int k = 0, a = 0; k < cnt; ++k) {
            const bool hit = a < n && ek[a] == k;
            part[(size_t)(k * 3 + 0) * d.Npad] = hit ? px[a] : 0.0;
            part[(size_t)(k * 3 + 1) * d.Npad] = hit ? py[a] : 0.0;
            part[(size_t)(k * 3 + 2) * d.Npad] = hit ? pz[a] : 0.0;
            if (hit) ++a;
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

__global__ void __launch_bounds__(kThreadsAtom) sw_force_kernel(Dev d, int p_lo) {
    int p;
    if (!image_of(blockIdx.y, p_lo, d.ctl->P, p)) return;
    const int slot = d.order[p];
    __shared__ double sh[9];
    __shared__ double red[32 * 7];
    if (threadIdx.x < 9) sh[threadIdx.x] = d.geom[slot].h[threadIdx.x];
    __syncthreads();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = i < d.N;
    const double rc2 = d.r_cut * d.r_cut;
    double fx = 0.0, fy = 0.0, fz = 0.0, vxx = 0.0, vyy = 0.0, vzz = 0.0, vxy = 0.0, vxz = 0.0, vyz = 0.0;
    if (valid) {
        const double4 *Rc = d.Rc + (size_t)slot * d.Npad;
        const uint32_t *lists = d.nbr_list + (size_t)slot * d.cap * d.Npad;
        const double *part = d.part + (size_t)slot * d.cap * 3 * d.Npad;
        const double4 ri = Rc[i];
        const int cnt = live_rows(d, slot, i);  // rows past it cannot be in range and are neither written nor read
        for (int k = 0; k < cnt; ++k) {
            const uint32_t e = lists[(size_t)k * d.Npad + i];
            const uint32_t j = e & kIdxMask, code = e >> kShiftBits;
            double dx, dy, dz;
            shifted_vec(ri, Rc[j], code, sh, dx, dy, dz);
            if (!(dx * dx + dy * dy + dz * dz < rc2)) continue;
            // mirror entry (j; i, -n): each 3-bit field n + 4 becomes 8 - (n + 4)
            const uint32_t rev = (uint32_t)i | ((((8u - (code & 7u)) & 7u) | (((8u - ((code >> 3) & 7u)) & 7u) << 3) |
                                                (((8u - ((code >> 6) & 7u)) & 7u) << 6)) << kShiftBits);
            const int l = d.nbr_mirror[((size_t)slot * d.cap + k) * d.Npad + i];  // row of (j; i, -n), found at the list build
            if (l >= d.cap || lists[(size_t)l * d.Npad + j] != rev) { set_error(d.ctl, CFNEB_EINVAL); continue; }
            const double gx = part[(size_t)(k * 3 + 0) * d.Npad + i] - part[(size_t)(l * 3 + 0) * d.Npad + j];  // Eq. 5
            const double gy = part[(size_t)(k * 3 + 1) * d.Npad + i] - part[(size_t)(l * 3 + 1) * d.Npad + j];
            const double gz = part[(size_t)(k * 3 + 2) * d.Npad + i] - part[(size_t)(l * 3 + 2) * d.Npad + j];
            fx += gx; fy += gy; fz += gz;
            vxx += dx * gx; vyy += dy * gy; vzz += dz * gz;  // Eq. 8; the total is symmetric, the halves are summed
            vxy += 0.5 * (dx * gy + dy * gx); vxz += 0.5 * (dx * gz + dz * gx); vyz += 0.5 * (dy * gz + dz * gy);
        }
        double *F = d.F + (size_t)slot * 3 * d.Npad;
        F[i] = fx; F[d.Npad + i] = fy; F[2 * (size_t)d.Npad + i] = fz;
    }
    double out7[7] = {0.0, -0.5 * vxx, -0.5 * vyy, -0.5 * vzz, -0.5 * vxy, -0.5 * vxz, -0.5 * vyz};
    block_sum<7>(out7, red);
    if (threadIdx.x == 0) {
        double *out = d.part_force + ((size_t)slot * d.nblk_force + blockIdx.x) * kNForcePart;
#pragma unroll
        for (int n = 0; n < 7; ++n) out[n] = out7[n];
        out[8] = 0.0;
    }
}

// Pass 2 for environments with many atoms inside the cut-off (descriptor network: 16 and more): U list rows per
// iteration, their loads issued together in two rounds (entries and mirror rows; then coordinates of j and both
// partial forces).  The walk is bound by the latency of these dependent gathers, not by bandwidth; a row past the
// count is replaced by row 0 and masked.  Measured at c6: 1.10 -> 1.00 ms per K2.  Where most live rows are outside
// the cut-off (Stillinger-Weber diamond: 4 of 5-16) the unconditional loads cost more than they hide (c5 0.50 ->
// 0.54 ms), and loading the partial forces in a third round after the range test loses the gain (c6 1.10, c5 0.52):
// that case keeps sw_force_kernel.
// ADD (the NEP-shaped potential): the rows that can lie inside the angular cut-off only, range test against it, and
// the result is added to F and to the virial partials that nep_radial_pair_kernel wrote before (same grid).
template <int U, bool ADD>
__global__ void __launch_bounds__(kThreadsAtom) pair_force_batched_kernel(Dev d, int p_lo) {
    int p;
    if (!image_of(blockIdx.y, p_lo, d.ctl->P, p)) return;
    const int slot = d.order[p];
    __shared__ double sh[9];
    __shared__ double red[32 * 7];
    if (threadIdx.x < 9) sh[threadIdx.x] = d.geom[slot].h[threadIdx.x];
    __syncthreads();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = i < d.N;
    const double rc2 = ADD ? d.pot[1] * d.pot[1] : d.r_cut * d.r_cut;
    double fx = 0.0, fy = 0.0, fz = 0.0, vxx = 0.0, vyy = 0.0, vzz = 0.0, vxy = 0.0, vxz = 0.0, vyz = 0.0;
    if (valid) {
        const double4 *Rc = d.Rc + (size_t)slot * d.Npad;
        const uint32_t *lists = d.nbr_list + (size_t)slot * d.cap * d.Npad;
        const double *part = d.part + (size_t)slot * d.cap * 3 * d.Npad;
        const double4 ri = Rc[i];
        // rows past it cannot be in range and are neither written nor read
        const int cnt = ADD ? nep_angular_rows(d, slot, i) : live_rows(d, slot, i);
        const unsigned short *mir = d.nbr_mirror + (size_t)slot * d.cap * d.Npad + i;
        for (int k0 = 0; k0 < cnt; k0 += U) {
            uint32_t e[U];
            int l[U];
            bool live[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                live[u] = k0 + u < cnt;
                const int k = live[u] ? k0 + u : 0;
                e[u] = lists[(size_t)k * d.Npad + i];
                l[u] = mir[(size_t)k * d.Npad];
            }
            double4 rj[U];
            double q[U][3], pp[U][3];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const uint32_t j = e[u] & kIdxMask;
                const int k = live[u] ? k0 + u : 0, lc = l[u] < d.cap ? l[u] : 0;
                rj[u] = Rc[j];
#pragma unroll
                for (int m = 0; m < 3; ++m) {
                    q[u][m] = part[(size_t)(lc * 3 + m) * d.Npad + j];
                    pp[u][m] = part[(size_t)(k * 3 + m) * d.Npad + i];
                }
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                double dx, dy, dz;
                shifted_vec(ri, rj[u], e[u] >> kShiftBits, sh, dx, dy, dz);
                if (!live[u] || !(dx * dx + dy * dy + dz * dz < rc2)) continue;
                if (l[u] >= d.cap) { set_error(d.ctl, CFNEB_EINVAL); continue; }  // no mirror entry (j; i, -n)
                const double gx = pp[u][0] - q[u][0], gy = pp[u][1] - q[u][1], gz = pp[u][2] - q[u][2];  // Eq. 5
                fx += gx; fy += gy; fz += gz;
                vxx += dx * gx; vyy += dy * gy; vzz += dz * gz;  // Eq. 8; the total is symmetric, the halves are summed
                vxy += 0.5 * (dx * gy + dy * gx); vxz += 0.5 * (dx * gz + dz * gx); vyz += 0.5 * (dy * gz + dz * gy);
            }
        }
        double *F = d.F + (size_t)slot * 3 * d.Npad;
        if (ADD) { fx += F[i]; fy += F[d.Npad + i]; fz += F[2 * (size_t)d.Npad + i]; }
        F[i] = fx; F[d.Npad + i] = fy; F[2 * (size_t)d.Npad + i] = fz;
    }
    double out7[7] = {0.0, -0.5 * vxx, -0.5 * vyy, -0.5 * vzz, -0.5 * vxy, -0.5 * vxz, -0.5 * vyz};
    block_sum<7>(out7, red);
    if (threadIdx.x == 0) {
        double *out = d.part_force + ((size_t)slot * d.nblk_force + blockIdx.x) * kNForcePart;
#pragma unroll
        for (int n = 0; n < 7; ++n) out[n] = ADD ? out[n] + out7[n] : out7[n];
        out[8] = 0.0;
    }
}

// After a list build: for every entry (i; j, n) the row of its mirror (j; i, -n) in j's list (cap if absent).
__global__ void __launch_bounds__(kThreadsAtom) sw_mirror_kernel(Dev d, int p_lo) {
    int p;
    if (!image_of(blockIdx.y, p_lo, d.ctl->P, p)) return;
    const int slot = d.order[p];
    if (!d.geom[slot].rebuild) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= d.N) return;
    const uint32_t *lists = d.nbr_list + (size_t)slot * d.cap * d.Npad;
    const int *counts = d.nbr_count + (size_t)slot * d.Npad;
    const int cnt = counts[i];
    for (int k = 0; k < cnt; ++k) {
        const uint32_t e = lists[(size_t)k * d.Npad + i];
        const uint32_t j = e & kIdxMask, code = e >> kShiftBits;
        const uint32_t rev = (uint32_t)i | ((((8u - (code & 7u)) & 7u) | (((8u - ((code >> 3) & 7u)) & 7u) << 3) |
                                            (((8u - ((code >> 6) & 7u)) & 7u) << 6)) << kShiftBits);
        const int cj = counts[j];
        int l = 0;
        while (l < cj && lists[(size_t)l * d.Npad + j] != rev) ++l;
        d.nbr_mirror[((size_t)slot * d.cap + k) * d.Npad + i] = (unsigned short)(l < cj ? l : d.cap);
    }
}

void launch_mirror_sw(const Dev &d, int p_lo, cudaStream_t st) {
    const int nimg = images_in_grid(d.S, p_lo);
    if (nimg <= 0) return;
    dim3 grid(d.nblk_atom, nimg);
    sw_mirror_kernel<<<grid, kThreadsAtom, 0, st>>>(d, p_lo);
}

void launch_pair_forces_manybody(const Dev &d, int p_lo, cudaStream_t st) {
    const int nimg = images_in_grid(d.S, p_lo);
    if (nimg <= 0) return;
    dim3 grid(d.nblk_atom, nimg);
    if (d.potential == CFNEB_POT_NEP) pair_force_batched_kernel<4, true><<<grid, kThreadsAtom, 0, st>>>(d, p_lo);
    else if (d.potential == CFNEB_POT_DNN) pair_force_batched_kernel<4, false><<<grid, kThreadsAtom, 0, st>>>(d, p_lo);
    else sw_force_kernel<<<grid, kThreadsAtom, 0, st>>>(d, p_lo);
}

void launch_force_sw(const Dev &d, int p_lo, cudaStream_t st) {
    const int nimg = images_in_grid(d.S, p_lo);
    if (nimg <= 0) return;
    dim3 grid(d.nblk_atom, nimg);
    sw_partial_kernel<<<grid, kThreadsAtom, 0, st>>>(d, p_lo);
    launch_pair_forces_manybody(d, p_lo, st);
}

}  // namespace cfn

// kernels_relax.cu -- cell-filter FIRE relaxation of the two endpoints on the device (
// BASELINE.json configs: "both endpoints cell-relaxed").  The same generalized coordinates and forces as the band
// (O0-O4: X = [R~ ; lam B], G = [F D^T ; D^-T V D^-1 / lam], Eq. 12, 17) with f = G -- no tangent, no springs -- and
// one FIRE state PER endpoint (O7 with n_rows = N + 3), i.e. two independent single-structure relaxations that
// share every launch.  K0-K2 and finalize_kernel run on the endpoint images only (p_lo = kEndpointsOnly); the three
// kernels here replace K4-K6:
//   relax_reduce_kernel   G.G, G.v, v.v and the max row norm of G over the atom rows (one pass over F, v)
//   relax_scalar_kernel   cell rows added; fmax = max row norm of G; freeze when fmax < tol (the oracle's loop
//                         tests convergence before every update); else the FIRE state machine -> cv, cf, sdt
//   relax_update_kernel   v <- cv v + cf G;  X <- X + sdt v  (both X buffers: endpoints are read from either)
#include "cfneb_internal.cuh"

namespace cfn {

constexpr int kNRelax = 4;  // GG, Gv, vv, max row norm^2

__device__ inline double2 ld2r(const double *p) { return *reinterpret_cast<const double2 *>(p); }
__device__ inline void st2r(double *p, double2 v) { *reinterpret_cast<double2 *>(p) = v; }

__global__ void __launch_bounds__(kThreadsStream) relax_reduce_kernel(Dev d) {
    const int e = blockIdx.y;
    const int slot = d.order[e ? d.ctl->P - 1 : 0];
    __shared__ double sD[9];
    __shared__ double red[32 * 3];
    __shared__ double redm[32];
    if (threadIdx.x < 9) sD[threadIdx.x] = d.geom[slot].D[threadIdx.x];
    __syncthreads();
    const size_t img = (size_t)3 * d.Npad;
    const double *F = d.F + slot * img, *V = d.v + slot * img;
    double acc[3] = {0.0, 0.0, 0.0}, m2 = 0.0;
    for (int tile = blockIdx.x; tile < d.nblk_stream; tile += gridDim.x) {
        const int i = 2 * (tile * kThreadsStream + threadIdx.x);
        if (i >= d.Npad) continue;
        double2 f[3], vv[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            f[c] = ld2r(F + (size_t)c * d.Npad + i);
            vv[c] = ld2r(V + (size_t)c * d.Npad + i);
        }
        double rx = 0.0, ry = 0.0;
#pragma unroll
        for (int c = 0; c < 3; ++c) {  // G = F D^T (Eq. 12)
            const double gx = f[0].x * sD[3 * c] + f[1].x * sD[3 * c + 1] + f[2].x * sD[3 * c + 2];
            const double gy = f[0].y * sD[3 * c] + f[1].y * sD[3 * c + 1] + f[2].y * sD[3 * c + 2];
            acc[0] += gx * gx + gy * gy;
            acc[1] += gx * vv[c].x + gy * vv[c].y;
            acc[2] += vv[c].x * vv[c].x + vv[c].y * vv[c].y;
            rx += gx * gx;
            ry += gy * gy;
        }
        m2 = fmax(m2, fmax(rx, ry));
    }
    block_sum<3>(acc, red);
    const double bm = block_max(m2, redm);
    if (threadIdx.x == 0) {
        double *out = d.part_relax + ((size_t)e * d.nblk_stream + blockIdx.x) * kNRelax;
        out[0] = acc[0]; out[1] = acc[1]; out[2] = acc[2]; out[3] = bm;
    }
}

// One thread per endpoint; partials summed in block order (bitwise repeatable).
__global__ void relax_scalar_kernel(Dev d, int nblk, double fmax_tol) {
    const int e = threadIdx.x;
    if (e >= 2) return;
    const int slot = d.order[e ? d.ctl->P - 1 : 0];
    RelaxState *rs = d.relax + e;
    double ff = 0.0, fv = 0.0, vv = 0.0, m2 = 0.0;
    const double *pr = d.part_relax + (size_t)e * d.nblk_stream * kNRelax;
    for (int b = 0; b < nblk; ++b) {
        ff += pr[b * kNRelax]; fv += pr[b * kNRelax + 1]; vv += pr[b * kNRelax + 2];
        m2 = fmax(m2, pr[b * kNRelax + 3]);
    }
    for (int r = 0; r < 3; ++r) {  // the three cell rows of the generalized vector
        double r2 = 0.0;
        for (int c = 0; c < 3; ++c) {
            const double g = d.Gc[slot * 9 + 3 * r + c], v = d.vc[slot * 9 + 3 * r + c];
            ff += g * g; fv += g * v; vv += v * v;
            r2 += g * g;
        }
        m2 = fmax(m2, r2);
    }
    const double fmax_now = sqrt(m2);
    rs->fmax = fmax_now;
    rs->E = d.E[slot];
    if (!isfinite(ff) || !isfinite(fv) || !isfinite(vv)) set_error(d.ctl, CFNEB_ENAN);
    if (rs->frozen || fmax_now < fmax_tol) {  // converged: this endpoint stops (oracle: `if fmax < tol: break`)
        rs->frozen = 1;
        rs->cv = 0.0; rs->cf = 0.0; rs->sdt = 0.0;
        return;
    }
    double dt = rs->dt, alpha = rs->alpha, cv, cf;
    int n_pos = rs->n_pos;
    if (rs->first) {  // A2
        rs->first = 0;
        cv = 0.0; cf = dt; vv = 0.0; fv = 0.0;
    } else if (fv > 0.0) {
        const double mix = (ff > 0.0) ? alpha * sqrt(vv / ff) : 0.0;
        cv = 1.0 - alpha;
        if (n_pos > d.fire_nmin) { dt = fmin(dt * d.finc, d.dtmax); alpha *= d.fa; }
        n_pos += 1;
        cf = mix + dt;
    } else {
        cv = 0.0; alpha = d.astart; dt *= d.fdec; n_pos = 0; cf = dt;
    }
    double vn2 = cv * cv * vv + 2.0 * cv * cf * fv + cf * cf * ff;
    if (vn2 < 0.0) vn2 = 0.0;
    const double nd = dt * sqrt(vn2), limit = d.maxstep * sqrt((double)(d.N + 3));  // A4 with n_rows = N + 3
    const double s = nd > limit ? limit / nd : 1.0;
    rs->dt = dt; rs->alpha = alpha; rs->n_pos = n_pos;
    rs->cv = cv; rs->cf = cf; rs->sdt = s * dt;
    rs->steps += 1;
}

__global__ void __launch_bounds__(kThreadsStream) relax_update_kernel(Dev d) {
    const int e = blockIdx.y;
    const int slot = d.order[e ? d.ctl->P - 1 : 0];
    const RelaxState *rs = d.relax + e;
    const double cv = rs->cv, cf = rs->cf, sdt = rs->sdt;
    if (rs->frozen) return;  // block-uniform
    __shared__ double sD[9];
    __shared__ double red[32];
    if (threadIdx.x < 9) sD[threadIdx.x] = d.geom[slot].D[threadIdx.x];
    __syncthreads();
    const size_t img = (size_t)3 * d.Npad, buf = (size_t)d.S * img;
    double *X = d.X + slot * img;
    const double *F = d.F + slot * img;
    double *V = d.v + slot * img;
    double v2max = 0.0;
    for (int tile = blockIdx.x; tile < d.nblk_stream; tile += gridDim.x) {
        const int i = 2 * (tile * kThreadsStream + threadIdx.x);
        if (i >= d.Npad) continue;
        double2 f[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) f[c] = ld2r(F + (size_t)c * d.Npad + i);
        double v2x = 0.0, v2y = 0.0;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const size_t o = (size_t)c * d.Npad + i;
            const double gx = f[0].x * sD[3 * c] + f[1].x * sD[3 * c + 1] + f[2].x * sD[3 * c + 2];
            const double gy = f[0].y * sD[3 * c] + f[1].y * sD[3 * c + 1] + f[2].y * sD[3 * c + 2];
            const double2 v0 = ld2r(V + o), x0 = ld2r(X + o);
            double2 vn, xn;
            vn.x = cv * v0.x + cf * gx; vn.y = cv * v0.y + cf * gy;
            xn.x = x0.x + sdt * vn.x;   xn.y = x0.y + sdt * vn.y;
            st2r(V + o, vn);
            st2r(X + o, xn);
            st2r(X + buf + o, xn);
            v2x += vn.x * vn.x; v2y += vn.y * vn.y;
        }
        v2max = fmax(v2max, fmax(v2x, v2y));
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        double xn[9];
        for (int k = 0; k < 9; ++k) {
            const double vn = cv * d.vc[slot * 9 + k] + cf * d.Gc[slot * 9 + k];
            d.vc[slot * 9 + k] = vn;
            xn[k] = d.Xc[slot * 9 + k] + sdt * vn;
        }
        if (d.cell_mode == CFNEB_CELL_B)  // O7 step 4: B <- (B + B^T)/2
            for (int r = 0; r < 3; ++r)
                for (int c = r + 1; c < 3; ++c) {
                    const double m = 0.5 * (xn[3 * r + c] + xn[3 * c + r]);
                    xn[3 * r + c] = m; xn[3 * c + r] = m;
                }
        for (int k = 0; k < 9; ++k) {
            d.Xc[slot * 9 + k] = xn[k];
            d.Xc[(size_t)d.S * 9 + slot * 9 + k] = xn[k];
        }
    }
    const double bd = block_max(sdt * sdt * v2max, red);
    if (threadIdx.x == 0) atomicMax(d.dispmax + slot, nonneg_bits(bd));
}

__global__ void relax_init_kernel(Dev d) {
    const int e = blockIdx.y;
    const int slot = d.order[e ? d.ctl->P - 1 : 0];
    const size_t img = (size_t)3 * d.Npad;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < img; i += (size_t)gridDim.x * blockDim.x)
        d.v[slot * img + i] = 0.0;
    if (blockIdx.x == 0 && threadIdx.x < 9) d.vc[slot * 9 + threadIdx.x] = 0.0;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        RelaxState *rs = d.relax + e;
        rs->dt = d.dt0; rs->alpha = d.astart; rs->cv = rs->cf = rs->sdt = 0.0;
        rs->fmax = 0.0; rs->E = 0.0;
        rs->n_pos = 0; rs->first = 1; rs->frozen = 0; rs->steps = 0;
    }
}

static int relax_blocks(const Dev &d) { return d.nblk_stream < 296 ? d.nblk_stream : 296; }

void launch_relax_init(const Dev &d, cudaStream_t st) {
    dim3 grid(64, 2);
    relax_init_kernel<<<grid, 256, 0, st>>>(d);
}

// one relaxation step of both endpoints after K0-K2 + finalize have run on them
void launch_relax_step(const Dev &d, double fmax_tol, cudaStream_t st) {
    const int nb = relax_blocks(d);
    dim3 grid(nb, 2);
    relax_reduce_kernel<<<grid, kThreadsStream, 0, st>>>(d);
    relax_scalar_kernel<<<1, 32, 0, st>>>(d, nb, fmax_tol);
    relax_update_kernel<<<grid, kThreadsStream, 0, st>>>(d);
}

}  // namespace cfn

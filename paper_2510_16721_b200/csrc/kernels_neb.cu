// kernels_neb.cu -- the band-level half of the iteration: K4 segmented reductions, K5 scalar kernel
// (improved tangent, climbing image, FIRE scalars), K6 fused NEB force + cell filter + FIRE update.
//
// Per movable image p with tau+ = X_{p+1} - X_p, tau- = X_p - X_{p-1} (generalized coordinates
// X = [R~ ; lam B], Eq. 17) and generalized force G = [F D^T ; D^-T V D^-1 / lam] (Eq. 12, 17):
//   tangent (ref [13])  tau = a tau+ + b tau-  with (a, b) chosen from E_{p-1}, E_p, E_{p+1}
//   Eq. 1           f = G - (G.t)t + k(|tau+| - |tau-|) t ,  t = tau/|tau|
//   climbing image (ref [12]) f = G - 2 (G.t) t
// Both have the form f = G + c1 tau+ + c2 tau- with per-image scalars c1, c2, so every band-level scalar
// FIRE needs (f.v, |f|, |v|, |v_new|) follows from ten dot products per image taken in ONE pass over
// X, F, v (K4); K6 then streams the same arrays once more and writes X_new, v_new.
#include "cfneb_internal.cuh"

namespace cfn {

__device__ inline double2 ld2(const double *p) { return *reinterpret_cast<const double2 *>(p); }
__device__ inline void st2(double *p, double2 v) { *reinterpret_cast<double2 *>(p) = v; }

// ------------------------------------------------------------------------------------------------
// K4: ten dot products over the atom rows of each movable image; per-block partials.
// grid (nblk_red, S-2), 256 threads.  An image is cut into nblk_stream tiles of 512 atoms (two atoms per thread,
// 128-bit loads on SoA rows); block b of an image takes tiles b, b + nblk_red, ... and keeps its ten sums in
// registers across tiles, so the shuffle / shared-memory reduction runs once per block instead of once per
// tile and loads of one block overlap the arithmetic of the others resident on the SM.  nblk_red is chosen so
// that the grid fills an integer number of waves (plan_stream_grids).  Blocks of neighbouring images work on
// the same tile index at about the same time, so X_{p-1} and X_{p+1} are L2 hits: DRAM sees X, F, v once (72 B).
constexpr int kThreadsReduce = 256, kBlocksReduce = 2;  // measured at c4: 6.07 TB/s; <256,3> spills (4.9), <128,5> spills (5.0)
template <int TR, int MINB, int UNROLL>
__global__ void __launch_bounds__(TR, MINB) reduce_kernel(Dev d) {
    const int p = blockIdx.y + 1;
    if (p > d.ctl->P - 2) return;
    const int sm = d.order[p - 1], s0 = d.order[p], sp = d.order[p + 1];
    __shared__ double sD[9];
    __shared__ double red[32 * kNDots];
    if (threadIdx.x < 9) sD[threadIdx.x] = d.geom[s0].D[threadIdx.x];
    __syncthreads();
    const size_t img = (size_t)3 * d.Npad;
    const double *Xb = d.X + (size_t)d.ctl->cur * d.S * img;
    const double *Xm = Xb + sm * img, *X0 = Xb + s0 * img, *Xp = Xb + sp * img;
    const double *F = d.F + s0 * img, *V = d.v + s0 * img;
    double acc[kNDots];
#pragma unroll
    for (int q = 0; q < kNDots; ++q) acc[q] = 0.0;
    const int ntile = (d.Npad + 2 * TR - 1) / (2 * TR);
    for (int tile = blockIdx.x; tile < ntile; tile += UNROLL * gridDim.x) {
        double2 f[UNROLL][3], xm[UNROLL][3], x0[UNROLL][3], xp[UNROLL][3], vv[UNROLL][3];
        bool on[UNROLL];
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
            const int t = tile + u * gridDim.x;
            const int i = 2 * (t * TR + threadIdx.x);
            on[u] = t < ntile && i < d.Npad;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const size_t o = (size_t)c * d.Npad + (on[u] ? i : 0);
                f[u][c] = on[u] ? ld2(F + o) : make_double2(0.0, 0.0);
                xm[u][c] = on[u] ? ld2(Xm + o) : make_double2(0.0, 0.0);
                x0[u][c] = on[u] ? ld2(X0 + o) : make_double2(0.0, 0.0);
                xp[u][c] = on[u] ? ld2(Xp + o) : make_double2(0.0, 0.0);
                vv[u][c] = on[u] ? ld2(V + o) : make_double2(0.0, 0.0);
            }
        }
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                // G = F D^T (Eq. 12): G_c = sum_m F_m D[c][m]
                const double gx = f[u][0].x * sD[3 * c] + f[u][1].x * sD[3 * c + 1] + f[u][2].x * sD[3 * c + 2];
                const double gy = f[u][0].y * sD[3 * c] + f[u][1].y * sD[3 * c + 1] + f[u][2].y * sD[3 * c + 2];
                const double tpx = xp[u][c].x - x0[u][c].x, tpy = xp[u][c].y - x0[u][c].y;
                const double tmx = x0[u][c].x - xm[u][c].x, tmy = x0[u][c].y - xm[u][c].y;
                acc[DOT_PP] += tpx * tpx + tpy * tpy;
                acc[DOT_MM] += tmx * tmx + tmy * tmy;
                acc[DOT_PM] += tpx * tmx + tpy * tmy;
                acc[DOT_GP] += gx * tpx + gy * tpy;
                acc[DOT_GM] += gx * tmx + gy * tmy;
                acc[DOT_GG] += gx * gx + gy * gy;
                acc[DOT_GV] += gx * vv[u][c].x + gy * vv[u][c].y;
                acc[DOT_PV] += tpx * vv[u][c].x + tpy * vv[u][c].y;
                acc[DOT_MV] += tmx * vv[u][c].x + tmy * vv[u][c].y;
                acc[DOT_VV] += vv[u][c].x * vv[u][c].x + vv[u][c].y * vv[u][c].y;
            }
        }
    }
    block_sum<kNDots>(acc, red);
    if (threadIdx.x == 0) {
        double *out = d.part_dots + ((size_t)s0 * d.nblk_stream + blockIdx.x) * kNDots;
#pragma unroll
        for (int q = 0; q < kNDots; ++q) out[q] = acc[q];
    }
}

// Second stage of K2 / K3, one block per image: E, V from the force partials (+ the pressure terms);
// G_cell (Eq. 17 / Eq. 14).  Fixed summation order (bitwise repeatable).  Does not depend on K4.
__global__ void __launch_bounds__(256) finalize_kernel(Dev d, int p_lo) {
    const int P = d.ctl->P;
    int p;
    if (!image_of(blockIdx.x, p_lo, P, p)) return;
    const int slot = d.order[p];
    __shared__ double red[32 * 8];
    double a8[8];  // [1..6] the virial; [0], [7] unused here (the energy channels go through two doubles)
#pragma unroll
    for (int q = 0; q < 8; ++q) a8[q] = 0.0;
    double e_hi = 0.0, e_lo = 0.0;
    const double *pf = d.part_force + (size_t)slot * d.nblk_force * kNForcePart;
    for (int b = threadIdx.x; b < d.nblk_force; b += blockDim.x) {
        const double *q8 = pf + (size_t)b * kNForcePart;
#pragma unroll
        for (int q = 1; q < 7; ++q) a8[q] += q8[q];
        dd_add(e_hi, e_lo, q8[0], q8[8]);  // pair energy, then site (embedding / many-body) energy of the block
        dd_add(e_hi, e_lo, q8[7], q8[9]);
    }
    block_sum<8>(a8, red);
    block_sum_dd(e_hi, e_lo, red);
    if (threadIdx.x == 0) {
        const Geom *g = d.geom + slot;
        // external pressure (A25): enthalpy H = U + p Omega and its virial V - p Omega I (Eq. 2-3)
        const double pv = d.pressure * fabs(g->vol);
        dd_add(e_hi, e_lo, pv, 0.0);
        const double E = e_hi + e_lo;
        const double V[9] = {a8[1] - pv, a8[4], a8[5], a8[4], a8[2] - pv, a8[6], a8[5], a8[6], a8[3] - pv};
        d.E[slot] = E;
        double Gc[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
        if (d.cell_mode != CFNEB_CELL_FIXED) {
            double T[9];
            mul3_atb(g->Dinv, V, T);  // D^-T V   (Eq. 13-14)
            if (d.cell_mode == CFNEB_CELL_B) mul3(T, g->Dinv, Gc);  // D^-T V D^-1 (Eq. 16-17, as printed)
            else for (int k = 0; k < 9; ++k) Gc[k] = T[k];
            for (int k = 0; k < 9; ++k) Gc[k] /= d.lam;
        }
        for (int k = 0; k < 9; ++k) {
            d.V[slot * 9 + k] = V[k];
            d.Gc[slot * 9 + k] = Gc[k];
        }
        if (!isfinite(E)) set_error(d.ctl, CFNEB_ENAN);
    }
}

// ------------------------------------------------------------------------------------------------
// K5: one block.  Tangent weights and c1, c2 per image in parallel; band totals and the FIRE state
// machine (O7: one state for the whole band, readings A1-A4) by thread 0 in path order.
__global__ void __launch_bounds__(1024) scalar_kernel(Dev d, int dry) {
    Ctl *ctl = d.ctl;
    const int P = ctl->P;
    __shared__ int s_pstar;
    {   // second stage of K4, one warp per image: the block partials of reduce_kernel summed in a fixed order
        // (lane-strided, then a shuffle tree), completed with the three cell rows of the generalized vectors
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
        const double *Xc = d.Xc + (size_t)ctl->cur * d.S * 9;
        for (int p = 1 + warp; p <= P - 2; p += nwarp) {
            const int slot = d.order[p];
            double a10[kNDots];
#pragma unroll
            for (int q = 0; q < kNDots; ++q) a10[q] = 0.0;
            const double *pd = d.part_dots + (size_t)slot * d.nblk_stream * kNDots;
            for (int b = lane; b < d.nblk_red; b += 32)
#pragma unroll
                for (int q = 0; q < kNDots; ++q) a10[q] += pd[(size_t)b * kNDots + q];
            if (lane < 9) {  // the nine cell components, one per lane
                const int sm = d.order[p - 1], sp = d.order[p + 1], k = lane;
                const double tp = Xc[sp * 9 + k] - Xc[slot * 9 + k], tm = Xc[slot * 9 + k] - Xc[sm * 9 + k];
                const double g = d.Gc[slot * 9 + k], v = d.vc[slot * 9 + k];
                a10[DOT_PP] += tp * tp; a10[DOT_MM] += tm * tm; a10[DOT_PM] += tp * tm;
                a10[DOT_GP] += g * tp;  a10[DOT_GM] += g * tm;  a10[DOT_GG] += g * g;
                a10[DOT_GV] += g * v;   a10[DOT_PV] += tp * v;  a10[DOT_MV] += tm * v;  a10[DOT_VV] += v * v;
            }
#pragma unroll
            for (int q = 0; q < kNDots; ++q)
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) a10[q] += __shfl_down_sync(0xffffffffu, a10[q], o);
            if (lane == 0)
                for (int q = 0; q < kNDots; ++q) d.dots[slot * kNDots + q] = a10[q];
        }
        __syncthreads();
    }
    __shared__ int s_pmax;
    if (threadIdx.x < 32) {  // argmax of the interior energies, lowest index on an exact tie: warp 0, lane-strided
        const int lane = threadIdx.x;
        int pb = -1;
        double best = 0.0;
        for (int p = 1 + lane; p <= P - 2; p += 32) {
            const double e = d.E[d.order[p]];
            if (pb < 0 || e > best) { best = e; pb = p; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double e2 = __shfl_down_sync(0xffffffffu, best, o);
            const int p2 = __shfl_down_sync(0xffffffffu, pb, o);
            if (p2 >= 0 && (pb < 0 || e2 > best || (e2 == best && p2 < pb))) { best = e2; pb = p2; }
        }
        if (lane == 0) {
            s_pmax = pb;
            s_pstar = d.climb ? pb : -1;  // climbing image (ref [12])
        }
    }
    __syncthreads();
    const int pstar = s_pstar;
    for (int p = 1 + threadIdx.x; p <= P - 2; p += blockDim.x) {
        const int slot = d.order[p];
        const double Em = d.E[d.order[p - 1]], E0 = d.E[slot], Ep = d.E[d.order[p + 1]];
        const double *dt = d.dots + slot * kNDots;
        double a, b;  // tau = a tau+ + b tau-   (improved tangent, ref [13])
        if (Ep > E0 && E0 > Em) { a = 1.0; b = 0.0; }
        else if (Ep < E0 && E0 < Em) { a = 0.0; b = 1.0; }
        else {
            const double dp = fabs(Ep - E0), dm = fabs(Em - E0);
            const double dmax = fmax(dp, dm), dmin = fmin(dp, dm);
            if (dmax == 0.0) { a = 1.0; b = 1.0; }  // A26: three equal energies, the weights vanish: bisector
            else if (Ep > Em) { a = dmax; b = dmin; } else { a = dmin; b = dmax; }
        }
        const double t2 = a * a * dt[DOT_PP] + 2.0 * a * b * dt[DOT_PM] + b * b * dt[DOT_MM];
        double c1 = 0.0, c2 = 0.0;
        if (!(t2 > 0.0)) set_error(ctl, isfinite(t2) ? CFNEB_EINVAL : CFNEB_ENAN);
        else {
            const double nt = sqrt(t2);
            const double Gt = (a * dt[DOT_GP] + b * dt[DOT_GM]) / nt;  // G . t^
            double coef;
            if (p == pstar) coef = -2.0 * Gt;
            else coef = -Gt + d.k_spring * (sqrt(dt[DOT_PP]) - sqrt(dt[DOT_MM]));
            c1 = coef * a / nt;
            c2 = coef * b / nt;
        }
        double *co = d.coef + slot * 4;
        co[0] = c1;
        co[1] = c2;
        co[2] = dt[DOT_GV] + c1 * dt[DOT_PV] + c2 * dt[DOT_MV];  // f . v
        co[3] = dt[DOT_GG] + c1 * c1 * dt[DOT_PP] + c2 * c2 * dt[DOT_MM] +
                2.0 * (c1 * dt[DOT_GP] + c2 * dt[DOT_GM] + c1 * c2 * dt[DOT_PM]);  // f . f
    }
    __syncthreads();
    if (threadIdx.x >= 32) return;
    // band totals: warp 0, lane-strided partial sums in path order, then a fixed shuffle tree
    double fv = 0.0, ff = 0.0, vv = 0.0, len = 0.0;
    {
        const int lane = threadIdx.x;
        for (int p = 1 + lane; p <= P - 2; p += 32) {
            const int slot = d.order[p];
            fv += d.coef[slot * 4 + 2];
            ff += d.coef[slot * 4 + 3];
            vv += d.dots[slot * kNDots + DOT_VV];
            len += sqrt(d.dots[slot * kNDots + DOT_PP]);
            if (p == 1) len += sqrt(d.dots[slot * kNDots + DOT_MM]);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            fv += __shfl_down_sync(0xffffffffu, fv, o);
            ff += __shfl_down_sync(0xffffffffu, ff, o);
            vv += __shfl_down_sync(0xffffffffu, vv, o);
            len += __shfl_down_sync(0xffffffffu, len, o);
        }
        if (lane != 0) return;
    }
    if (ff < 0.0) ff = 0.0;  // round-off of the one-pass algebra near convergence
    if (!isfinite(fv) || !isfinite(ff) || !isfinite(vv)) set_error(ctl, CFNEB_ENAN);
    ctl->pstar = pstar;
    ctl->path_length = len;
    {
        const int pb = s_pmax;
        ctl->barrier = (pb > 0) ? d.E[d.order[pb]] - d.E[d.order[0]] : 0.0;
    }
    if (dry) return;
    if (ctl->steps > 0ull) {  // per-step record: the previous iteration's max row norm^2, complete now that its K6 has run
        double f2;
        const unsigned long long b = ctl->fmax_bits;
        memcpy(&f2, &b, sizeof f2);
        d.hist[((ctl->steps - 1ull) % kHistLen) * kHistFields + 1] = f2;
    }
    ctl->fmax_bits = 0ull;  // K6 of this step takes the max row norm of f (O8)
    // ---- FIRE (O7) ----
    double dt = ctl->dt, alpha = ctl->alpha, cv, cf;
    int n_pos = ctl->n_pos;
    if (ctl->first) {  // A2: no power test on the first step after a (re)start; v = 0
        ctl->first = 0;
        cv = 0.0;
        cf = dt;
        vv = 0.0;
        fv = 0.0;
    } else if (fv > 0.0) {
        const double mix = (ff > 0.0) ? alpha * sqrt(vv / ff) : 0.0;  // alpha |v| / |f|
        cv = 1.0 - alpha;
        if (n_pos > d.fire_nmin) {
            dt = fmin(dt * d.finc, d.dtmax);
            alpha *= d.fa;
        }
        n_pos += 1;
        cf = mix + dt;
    } else {
        cv = 0.0;
        alpha = d.astart;
        dt *= d.fdec;
        n_pos = 0;
        cf = dt;
    }
    // |v_new|^2 with v_new = cv v + cf f;  Delta = dt v_new, limited to maxstep sqrt(movable rows) (A4)
    double vn2 = cv * cv * vv + 2.0 * cv * cf * fv + cf * cf * ff;
    if (vn2 < 0.0) vn2 = 0.0;
    const double nd = dt * sqrt(vn2);
    const double limit = d.maxstep * sqrt((double)(P - 2) * (double)(d.N + 3));
    double s = 1.0;
    if (nd > limit) s = limit / nd;
    ctl->dt = dt;
    ctl->alpha = alpha;
    ctl->n_pos = n_pos;
    ctl->cv = cv;
    ctl->cf = cf;
    ctl->sdt = s * dt;
    ctl->src = ctl->cur;
    ctl->dst = 1 - ctl->cur;
    ctl->cur = 1 - ctl->cur;
    {   // per-step record (cfneb_get_history): what cfneb_get_status would report after this iteration, except its
        // fmax, which K6 is about to produce (filed by the next K5, or read from the control block for the last one)
        double *row = d.hist + (ctl->steps % kHistLen) * kHistFields;
        row[0] = (double)(ctl->steps + 1ull);
        row[1] = 0.0;
        row[2] = ctl->barrier;
        row[3] = (double)pstar;
        row[4] = dt;
        row[5] = alpha;
        row[6] = (double)P;
        row[7] = (double)ctl->rebuilds;
    }
    ctl->steps += 1ull;
}

void launch_reduce(const Dev &d, cudaStream_t st) {
    if (d.S < 3) return;
    dim3 grid(d.nblk_red, d.S - 2);
    reduce_kernel<kThreadsReduce, kBlocksReduce, 1><<<grid, kThreadsReduce, 0, st>>>(d);
}

// Blocks per image for a streaming kernel that keeps `occ` blocks resident per SM: the smallest whole number
// of waves w for which floor(w * slots / M) blocks per image fill >= 95 % of the w * slots block slots
// (M = S - 2 images), never more than one block per tile.
static int blocks_per_image(int tiles, int images, int slots) {
    if (images < 1) return 1;
    int best = 1;
    double best_fill = 0.0;
    for (int w = 1; w <= 8; ++w) {
        int b = (w * slots) / images;
        if (b < 1) continue;
        if (b >= tiles) return tiles;
        const double fill = (double)b * images / ((double)w * slots);
        if (fill > best_fill + 1e-9) { best_fill = fill; best = b; }
        if (fill >= 0.95) break;
    }
    return best < tiles ? best : tiles;
}

int update_blocks_per_sm();  // kernels_update.cu

void plan_stream_grids(Dev &d) {
    int dev = 0, sms = 148, occ_r = 3, occ_u = 2;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    // measured on B200 at c4 (profiles/): reduce <2 blocks/SM, 1 tile in flight> 5.5 TB/s (114 registers, no spill;
    // <3, 1> spills and reaches 4.9, <2, 2> 4.8); update <3 blocks/SM> 6.2 TB/s (76 registers; <2> 5.9)
    occ_r = kBlocksReduce;
    occ_u = update_blocks_per_sm();
    d.nblk_red = blocks_per_image((d.Npad + 2 * kThreadsReduce - 1) / (2 * kThreadsReduce), d.S - 2, sms * occ_r);
    if (d.nblk_red > d.nblk_stream) d.nblk_red = d.nblk_stream;  // part_dots holds nblk_stream rows per image
    d.nblk_upd = blocks_per_image(d.nblk_stream, d.S - 2, sms * occ_u);
}

void launch_finalize(const Dev &d, int p_lo, cudaStream_t st) {
    const int nimg = images_in_grid(d.S, p_lo);
    if (nimg <= 0) return;
    finalize_kernel<<<nimg, 256, 0, st>>>(d, p_lo);
}

void launch_scalar(const Dev &d, int dry, cudaStream_t st) { scalar_kernel<<<1, 1024, 0, st>>>(d, dry); }

}  // namespace cfn

// kernels_adapt.cu -- O9 (adaptive image control, "the image distribution is automatically adjusted"; reading
// A16) decided and applied on the device, so that a run with adaptive insertion / deletion needs no host round
// trip either.  Same rule as the host path cfneb_adapt: per control step at most one
// deletion (the interior, non-climbing image q minimising d_{q-1} + d_q, if below d_delete and P > 3), then at most
// one insertion (midpoint of the longest segment, if above d_insert and a slot is free); FIRE restarts after any
// change.  The order table, P, the free-slot stack and the climbing index live in device memory; the host mirrors
// are refreshed lazily by the next call that needs them.
//
// Enqueued sequence (every kernel exits at once when it has nothing to do):
//   segment_lengths -> adapt_delete -> segment_lengths -> adapt_insert -> adapt_midpoint -> adapt_reset_fire
#include "cfneb_internal.cuh"

namespace cfn {

__global__ void adapt_delete_kernel(Dev d, const double *__restrict__ seglen, double d_delete) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    Ctl *c = d.ctl;
    c->changed = 0;
    c->ins_new = -1;
    const int P = c->P;
    if (P <= 3) return;
    int best = -1;
    double bs = 0.0;
    for (int q = 1; q <= P - 2; ++q) {
        if (q == c->pstar) continue;
        const double s = seglen[q - 1] + seglen[q];
        if (best < 0 || s < bs) { best = q; bs = s; }
    }
    if (best > 0 && bs < d_delete) {
        d.free_stack[c->n_free] = d.order[best];
        c->n_free += 1;
        for (int q = best; q < P - 1; ++q) d.order[q] = d.order[q + 1];
        c->P = P - 1;
        if (c->pstar > best) c->pstar -= 1;  // the reported climbing index stays on the same image
        c->changed = 1;
        c->n_deleted += 1;
    }
}

__global__ void adapt_insert_kernel(Dev d, const double *__restrict__ seglen, double d_insert) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    Ctl *c = d.ctl;
    const int P = c->P;
    int q = 0;
    for (int k = 1; k <= P - 2; ++k)
        if (seglen[k] > seglen[q]) q = k;
    if (seglen[q] > d_insert && P < d.S && c->n_free > 0) {
        c->n_free -= 1;
        const int sn = d.free_stack[c->n_free];
        c->ins_a = d.order[q];
        c->ins_b = d.order[q + 1];
        c->ins_new = sn;
        for (int k = P; k > q + 1; --k) d.order[k] = d.order[k - 1];
        d.order[q + 1] = sn;
        c->P = P + 1;
        if (c->pstar > q) c->pstar += 1;
        c->changed = 1;
        c->n_inserted += 1;
    }
}

// K7 with its operands read from the control block (set by adapt_insert_kernel)
__global__ void adapt_midpoint_kernel(Dev d) {
    const int sn = d.ctl->ins_new;
    if (sn < 0) return;
    const int sa = d.ctl->ins_a, sb = d.ctl->ins_b;
    const size_t img = (size_t)3 * d.Npad, buf = (size_t)d.S * img;
    const double *Xs = d.X + (size_t)d.ctl->cur * buf;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < img; i += (size_t)gridDim.x * blockDim.x) {
        const double x = 0.5 * (Xs[sa * img + i] + Xs[sb * img + i]);
        d.X[sn * img + i] = x;
        d.X[buf + sn * img + i] = x;
        d.v[sn * img + i] = 0.0;
        d.F[sn * img + i] = 0.0;
    }
    if (blockIdx.x == 0 && threadIdx.x < 9) {
        const double *Xc = d.Xc + (size_t)d.ctl->cur * d.S * 9;
        const double x = 0.5 * (Xc[sa * 9 + threadIdx.x] + Xc[sb * 9 + threadIdx.x]);
        d.Xc[sn * 9 + threadIdx.x] = x;
        d.Xc[(size_t)d.S * 9 + sn * 9 + threadIdx.x] = x;
        d.vc[sn * 9 + threadIdx.x] = 0.0;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        d.E[sn] = __longlong_as_double(0x7ff8000000000000ll);  // NaN until the next evaluation
        Geom *g = d.geom + sn;
        g->force_rebuild = 1;
        g->acc = 0.0;
        g->since = 0;
        d.dispmax[sn] = 0ull;
        d.dispmax_in[sn] = 0ull;
    }
}

__global__ void adapt_reset_fire_kernel(Dev d) {
    if (!d.ctl->changed) return;
    const size_t n = (size_t)d.S * 3 * d.Npad;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) d.v[i] = 0.0;
    if (blockIdx.x == 0) {
        for (int k = threadIdx.x; k < d.S * 9; k += blockDim.x) d.vc[k] = 0.0;
        if (threadIdx.x == 0) {
            Ctl *c = d.ctl;
            c->dt = d.dt0;
            c->alpha = d.astart;
            c->n_pos = 0;
            c->first = 1;
        }
    }
}

// ------------------------------------------------------------------------------------------------------------------
// Arc-length re-parametrisation ("the image distribution is automatically adjusted ... based on local spacing in
// configuration space"; reading A27): the interior images are moved to equal arc length along the band's own polyline
// in X.  With s_p = sum_{q<p} |X_{q+1} - X_q|, image p goes to the point at arc length p L / (P - 1) on the segment
// that contains it; with hold_climbing the climbing image stays and each side is redistributed on its own.  Three
// kernels on the stream, nothing read back:  segment_lengths -> reparam_plan (one thread: the running sums, in path
// order) -> reparam_apply (every image written into the other coordinate buffer from the untouched current one; the
// largest atomic displacement of each image goes into the staleness bound of its neighbour list) -> reparam_commit
// (buffer flip, FIRE restart as after any O9 change).
__global__ void reparam_plan_kernel(Dev d, const double *__restrict__ seglen, int hold_climbing) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const Ctl *c = d.ctl;
    const int P = c->P;
    int knots[3] = {0, P - 1, P - 1}, nk = 2;
    if (hold_climbing && d.climb && c->pstar > 0 && c->pstar < P - 1) { knots[1] = c->pstar; nk = 3; }
    double *s = d.seglen + d.S;  // second half of the seglen buffer: s_p, p = 0..P-1
    s[0] = 0.0;
    for (int p = 1; p < P; ++p) s[p] = s[p - 1] + seglen[p - 1];
    for (int p = 0; p < P; ++p) { d.plan_q[p] = p; d.plan_t[p] = 0.0; }
    for (int kk = 0; kk + 1 < nk; ++kk) {
        const int lo = knots[kk], hi = knots[kk + 1];
        for (int p = lo + 1; p < hi; ++p) {
            const double target = s[lo] + (s[hi] - s[lo]) * (double)(p - lo) / (double)(hi - lo);
            int q = lo;
            while (q < hi - 1 && s[q + 1] <= target) ++q;  // segment q with s_q <= target < s_{q+1}
            d.plan_q[p] = q;
            d.plan_t[p] = s[q + 1] > s[q] ? (target - s[q]) / (s[q + 1] - s[q]) : 0.0;
        }
    }
}

__global__ void __launch_bounds__(256) reparam_apply_kernel(Dev d) {
    const int p = blockIdx.y;
    const int P = d.ctl->P;
    if (p >= P) return;
    const int q = d.plan_q[p];
    const double t = d.plan_t[p];
    const int slot = d.order[p], sa = d.order[q], sb = d.order[min(q + 1, P - 1)];
    const size_t img = (size_t)3 * d.Npad, buf = (size_t)d.S * img;
    const int cur = d.ctl->cur;
    const double *Xs = d.X + (size_t)cur * buf;
    double *Xd = d.X + (size_t)(1 - cur) * buf;
    __shared__ double red[32];
    double d2 = 0.0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < d.Npad; i += gridDim.x * blockDim.x) {
        double dd = 0.0;
        for (int c = 0; c < 3; ++c) {
            const size_t o = (size_t)c * d.Npad + i;
            const double a = Xs[sa * img + o];
            const double x = t == 0.0 ? a : a + t * (Xs[sb * img + o] - a);
            const double dx = x - Xs[slot * img + o];
            dd += dx * dx;
            Xd[slot * img + o] = x;
        }
        d2 = fmax(d2, dd);
    }
    if (!(d2 == d2)) d2 = 1e300;
    const double bm = block_max(d2, red);
    if (threadIdx.x == 0) atomicMax(d.dispmax_in + slot, nonneg_bits(bm));
    if (blockIdx.x == 0 && threadIdx.x < 9) {
        const double *Xc = d.Xc + (size_t)cur * d.S * 9;
        const int k = threadIdx.x;
        const double a = Xc[sa * 9 + k];
        double x = t == 0.0 ? a : a + t * (Xc[sb * 9 + k] - a);
        if (d.cell_mode == CFNEB_CELL_B && t != 0.0) {  // B <- 1/2 (B + B^T), as after every update (O7 step 4)
            const int kt = 3 * (k % 3) + k / 3;
            const double at = Xc[sa * 9 + kt];
            x = 0.5 * (x + (at + t * (Xc[sb * 9 + kt] - at)));
        }
        d.Xc[(size_t)(1 - cur) * d.S * 9 + slot * 9 + k] = x;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0 && (t != 0.0 || q != p))
        d.E[slot] = __longlong_as_double(0x7ff8000000000000ll);  // a moved image: NaN until the next evaluation
}

__global__ void reparam_commit_kernel(Dev d) {
    const size_t n = (size_t)d.S * 3 * d.Npad;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) d.v[i] = 0.0;
    if (blockIdx.x == 0) {
        for (int k = threadIdx.x; k < d.S * 9; k += blockDim.x) d.vc[k] = 0.0;
        if (threadIdx.x == 0) {
            Ctl *c = d.ctl;
            c->cur = 1 - c->cur;
            c->dt = d.dt0;
            c->alpha = d.astart;
            c->n_pos = 0;
            c->first = 1;
        }
    }
}

void launch_reparametrize(const Dev &d, int hold_climbing, cudaStream_t st) {
    launch_segment_lengths(d, d.seglen, st);
    reparam_plan_kernel<<<1, 32, 0, st>>>(d, d.seglen, hold_climbing);
    int bx = (d.Npad + 255) / 256;
    if (bx > 64) bx = 64;
    dim3 grid(bx, d.S);
    launch_pending_guard(d, 0, d.S, st);  // an earlier move not yet seen by K0: its displacement adds to this one
    reparam_apply_kernel<<<grid, 256, 0, st>>>(d);
    reparam_commit_kernel<<<592, 256, 0, st>>>(d);
}

void launch_adapt_device(const Dev &d, double d_insert, double d_delete, cudaStream_t st) {
    launch_segment_lengths(d, d.seglen, st);
    adapt_delete_kernel<<<1, 32, 0, st>>>(d, d.seglen, d_delete);
    launch_segment_lengths(d, d.seglen, st);
    adapt_insert_kernel<<<1, 32, 0, st>>>(d, d.seglen, d_insert);
    adapt_midpoint_kernel<<<296, 256, 0, st>>>(d);
    adapt_reset_fire_kernel<<<592, 256, 0, st>>>(d);
}

}  // namespace cfn

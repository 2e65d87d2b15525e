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

void launch_adapt_device(const Dev &d, double d_insert, double d_delete, cudaStream_t st) {
    launch_segment_lengths(d, d.seglen, st);
    adapt_delete_kernel<<<1, 32, 0, st>>>(d, d.seglen, d_delete);
    launch_segment_lengths(d, d.seglen, st);
    adapt_insert_kernel<<<1, 32, 0, st>>>(d, d.seglen, d_insert);
    adapt_midpoint_kernel<<<296, 256, 0, st>>>(d);
    adapt_reset_fire_kernel<<<592, 256, 0, st>>>(d);
}

}  // namespace cfn

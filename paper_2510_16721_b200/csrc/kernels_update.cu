// kernels_update.cu -- K6: fused NEB-force assembly (Eq. 1) + cell-filter transform (Eq. 12, 17) + FIRE
// update, streaming X_{p-1}, X_p, X_{p+1}, F, v once and writing X_new, v_new; K7 image interpolation for
// insertion; the export kernels behind the parity / checkpoint hooks.
#include "cfneb_internal.cuh"

namespace cfn {

__device__ inline double2 ld2(const double *p) { return *reinterpret_cast<const double2 *>(p); }
__device__ inline void st2(double *p, double2 v) { *reinterpret_cast<double2 *>(p) = v; }

// grid (nblk_upd, S-2), 256 threads, two atoms per thread and tile; block b of an image takes the 512-atom tiles
// b, b + nblk_upd, ... (same tiling as K4, see reduce_kernel).
//   f = F D^T + c1 tau+ + c2 tau-          (c1, c2 from K5: perpendicular projection + spring / climbing)
//   v_new = cv v + cf f ;  X_new = X + sdt v_new     (cv, cf, sdt from K5: FIRE mixing, dt, step clip)
// Also: max row norm of f (fmax, O8) and max |dR~_i|^2 of this image (neighbour-list skin test of K0).
template <int MINB>
__global__ void __launch_bounds__(kThreadsStream, MINB) update_kernel(Dev d) {
    const int p = blockIdx.y + 1;
    const Ctl *ctl = d.ctl;
    if (p > ctl->P - 2) return;
    const int sm = d.order[p - 1], s0 = d.order[p], sp = d.order[p + 1];
    __shared__ double sD[9];
    __shared__ double red[32];
    if (threadIdx.x < 9) sD[threadIdx.x] = d.geom[s0].D[threadIdx.x];
    __syncthreads();
    const double c1 = d.coef[s0 * 4], c2 = d.coef[s0 * 4 + 1];
    const double cv = ctl->cv, cf = ctl->cf, sdt = ctl->sdt;
    const size_t img = (size_t)3 * d.Npad;
    const double *Xs = d.X + (size_t)ctl->src * d.S * img;
    double *Xd = d.X + (size_t)ctl->dst * d.S * img + s0 * img;
    const double *Xm = Xs + sm * img, *X0 = Xs + s0 * img, *Xp = Xs + sp * img;
    const double *F = d.F + s0 * img;
    double *V = d.v + s0 * img;
    double f2max = 0.0, v2max = 0.0;
    for (int tile = blockIdx.x; tile < d.nblk_stream; tile += gridDim.x) {
        const int i = 2 * (tile * kThreadsStream + threadIdx.x);
        if (i >= d.Npad) continue;
        double2 f[3], xm[3], x0[3], xp[3], vv[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const size_t o = (size_t)c * d.Npad + i;
            f[c] = ld2(F + o);
            xm[c] = ld2(Xm + o);
            x0[c] = ld2(X0 + o);
            xp[c] = ld2(Xp + o);
            vv[c] = ld2(V + o);
        }
        double f2x = 0.0, f2y = 0.0, v2x = 0.0, v2y = 0.0;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double gx = f[0].x * sD[3 * c] + f[1].x * sD[3 * c + 1] + f[2].x * sD[3 * c + 2];
            const double gy = f[0].y * sD[3 * c] + f[1].y * sD[3 * c + 1] + f[2].y * sD[3 * c + 2];
            const double fx = gx + c1 * (xp[c].x - x0[c].x) + c2 * (x0[c].x - xm[c].x);
            const double fy = gy + c1 * (xp[c].y - x0[c].y) + c2 * (x0[c].y - xm[c].y);
            double2 vn, xn;
            vn.x = cv * vv[c].x + cf * fx;
            vn.y = cv * vv[c].y + cf * fy;
            xn.x = x0[c].x + sdt * vn.x;
            xn.y = x0[c].y + sdt * vn.y;
            const size_t o = (size_t)c * d.Npad + i;
            st2(V + o, vn);
            st2(Xd + o, xn);
            f2x += fx * fx; f2y += fy * fy;
            v2x += vn.x * vn.x; v2y += vn.y * vn.y;
        }
        f2max = fmax(f2max, fmax(f2x, f2y));
        v2max = fmax(v2max, fmax(v2x, v2y));
    }
    const double d2max = sdt * sdt * v2max;
    // cell block (three rows of the generalized vector): block 0, thread 0 of every image
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        const double *Xcs = d.Xc + (size_t)ctl->src * d.S * 9;
        double *Xcd = d.Xc + (size_t)ctl->dst * d.S * 9 + s0 * 9;
        double xn[9];
        for (int r = 0; r < 3; ++r) {
            double f2 = 0.0;
            for (int c = 0; c < 3; ++c) {
                const int k = 3 * r + c;
                const double x = Xcs[s0 * 9 + k];
                const double fk = d.Gc[s0 * 9 + k] + c1 * (Xcs[sp * 9 + k] - x) + c2 * (x - Xcs[sm * 9 + k]);
                const double vn = cv * d.vc[s0 * 9 + k] + cf * fk;
                d.vc[s0 * 9 + k] = vn;
                xn[k] = x + sdt * vn;
                f2 += fk * fk;
            }
            f2max = fmax(f2max, f2);
        }
        if (d.cell_mode == CFNEB_CELL_B) {  // O7 step 4: B <- (B + B^T)/2
            for (int r = 0; r < 3; ++r)
                for (int c = r + 1; c < 3; ++c) {
                    const double m = 0.5 * (xn[3 * r + c] + xn[3 * c + r]);
                    xn[3 * r + c] = m;
                    xn[3 * c + r] = m;
                }
        }
        for (int k = 0; k < 9; ++k) Xcd[k] = xn[k];
    }
    const double bf = block_max(f2max, red);
    const double bd = block_max(d2max, red);
    if (threadIdx.x == 0) {
        atomicMax(&d.ctl->fmax_bits, nonneg_bits(bf));
        atomicMax(d.dispmax + s0, nonneg_bits(bd));
    }
}

// Parity hook: f^NEB of every image in the external layout fneb[p][(N+3)][3] (zero rows for endpoints),
// from the coefficients of a dry K5 at the current X.
__global__ void materialize_fneb_kernel(Dev d) {
    const int p = blockIdx.y;
    const int P = d.ctl->P;
    if (p >= P) return;
    const int rows = d.N + 3;
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= rows) return;
    double *out = d.fneb + ((size_t)p * rows + (a < d.N ? d.perm[a] : a)) * 3;
    if (p == 0 || p == P - 1) {
        out[0] = out[1] = out[2] = 0.0;
        return;
    }
    const int sm = d.order[p - 1], s0 = d.order[p], sp = d.order[p + 1];
    const double c1 = d.coef[s0 * 4], c2 = d.coef[s0 * 4 + 1];
    if (a < d.N) {
        const size_t img = (size_t)3 * d.Npad;
        const double *Xb = d.X + (size_t)d.ctl->cur * d.S * img;
        const double *D = d.geom[s0].D;
        const double *F = d.F + s0 * img;
        const double Fx = F[a], Fy = F[d.Npad + a], Fz = F[2 * (size_t)d.Npad + a];
        for (int c = 0; c < 3; ++c) {
            const size_t o = (size_t)c * d.Npad + a;
            const double x = Xb[s0 * img + o];
            const double g = Fx * D[3 * c] + Fy * D[3 * c + 1] + Fz * D[3 * c + 2];
            out[c] = g + c1 * (Xb[sp * img + o] - x) + c2 * (x - Xb[sm * img + o]);
        }
    } else {
        const double *Xc = d.Xc + (size_t)d.ctl->cur * d.S * 9;
        for (int c = 0; c < 3; ++c) {
            const int k = 3 * (a - d.N) + c;
            const double x = Xc[s0 * 9 + k];
            out[c] = d.Gc[s0 * 9 + k] + c1 * (Xc[sp * 9 + k] - x) + c2 * (x - Xc[sm * 9 + k]);
        }
    }
}

// Parity hook (cfneb_get_dots): the generalized force G = [F D^T ; G_cell] (Eq. 12, 17) of every image in the
// external layout [p][(N+3)][3] (zero rows for endpoints), written into the fneb buffer; and the K4 dot products and
// K5 coefficients of a dry evaluation in path order.
__global__ void materialize_gen_force_kernel(Dev d) {
    const int p = blockIdx.y;
    const int P = d.ctl->P;
    if (p >= P) return;
    const int rows = d.N + 3;
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= rows) return;
    double *out = d.fneb + ((size_t)p * rows + (a < d.N ? d.perm[a] : a)) * 3;
    if (p == 0 || p == P - 1) {
        out[0] = out[1] = out[2] = 0.0;
        return;
    }
    const int s0 = d.order[p];
    if (a < d.N) {
        const double *D = d.geom[s0].D;
        const double *F = d.F + (size_t)s0 * 3 * d.Npad;
        const double Fx = F[a], Fy = F[d.Npad + a], Fz = F[2 * (size_t)d.Npad + a];
        for (int c = 0; c < 3; ++c) out[c] = Fx * D[3 * c] + Fy * D[3 * c + 1] + Fz * D[3 * c + 2];
    } else {
        for (int c = 0; c < 3; ++c) out[c] = d.Gc[s0 * 9 + 3 * (a - d.N) + c];
    }
}

__global__ void export_dots_kernel(Dev d, double *dots_out, double *coef_out) {
    const int P = d.ctl->P;
    for (int i = threadIdx.x; i < P * kNDots; i += blockDim.x) {
        const int p = i / kNDots, q = i % kNDots;
        dots_out[i] = (p == 0 || p == P - 1) ? 0.0 : d.dots[d.order[p] * kNDots + q];
    }
    for (int i = threadIdx.x; i < P * 4; i += blockDim.x) {
        const int p = i / 4, q = i % 4;
        coef_out[i] = (p == 0 || p == P - 1) ? 0.0 : d.coef[d.order[p] * 4 + q];
    }
}

// K7: new image = midpoint of two stored images in generalized coordinates (O9); v = 0; energy unknown.
__global__ void midpoint_kernel(Dev d, int sa, int sb, int sn) {
    const size_t img = (size_t)3 * d.Npad, buf = (size_t)d.S * img;
    const double *Xs = d.X + (size_t)d.ctl->cur * buf;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < img) {
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
    }
}

// FIRE restart (O9: after any insertion / deletion): v = 0, dt = dt0, alpha = alpha_start, first = true.
__global__ void reset_fire_kernel(Dev d) {
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

// d_p = |X_{p+1} - X_p| over all (N+3) x 3 components, one block per segment (O8).
__global__ void __launch_bounds__(256) segment_lengths_kernel(Dev d, double *out) {
    const int p = blockIdx.x;
    if (p > d.ctl->P - 2) return;
    const int sa = d.order[p], sb = d.order[p + 1];
    __shared__ double red[32];
    const size_t img = (size_t)3 * d.Npad;
    const double *Xb = d.X + (size_t)d.ctl->cur * d.S * img;
    double acc[1] = {0.0};
    for (size_t i = threadIdx.x; i < img; i += blockDim.x) {
        const double t = Xb[sb * img + i] - Xb[sa * img + i];
        acc[0] += t * t;
    }
    if (threadIdx.x < 9) {
        const double *Xc = d.Xc + (size_t)d.ctl->cur * d.S * 9;
        const double t = Xc[sb * 9 + threadIdx.x] - Xc[sa * 9 + threadIdx.x];
        acc[0] += t * t;
    }
    block_sum<1>(acc, red);
    if (threadIdx.x == 0) out[p] = sqrt(acc[0]);
}

// ---- exports to the external row-major layouts (path order) ----
__global__ void export_path_kernel(Dev d, double *pos, double *cells, double *E) {
    const int p = blockIdx.y;
    if (p >= d.ctl->P) return;
    const int slot = d.order[p];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < d.N && pos) {
        const double4 r = d.Rc[(size_t)slot * d.Npad + i];
        double *o = pos + ((size_t)p * d.N + d.perm[i]) * 3;
        o[0] = r.x; o[1] = r.y; o[2] = r.z;
    }
    if (blockIdx.x == 0 && threadIdx.x < 9 && cells) cells[p * 9 + threadIdx.x] = d.geom[slot].h[threadIdx.x];
    if (blockIdx.x == 0 && threadIdx.x == 0 && E) E[p] = d.E[slot];
}

__global__ void export_state_kernel(Dev d, double *Xo, double *vo) {
    const int p = blockIdx.y;
    const int P = d.ctl->P;
    if (p >= P) return;
    const int slot = d.order[p];
    const int rows = d.N + 3;
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= rows) return;
    const size_t img = (size_t)3 * d.Npad;
    const double *Xb = d.X + ((size_t)d.ctl->cur * d.S + slot) * img;
    const double *Xc = d.Xc + ((size_t)d.ctl->cur * d.S + slot) * 9;
    const bool movable = p > 0 && p < P - 1;
    const int ao = a < d.N ? d.perm[a] : a;  // row of the caller's layout
    for (int c = 0; c < 3; ++c) {
        double x, v;
        if (a < d.N) {
            x = Xb[(size_t)c * d.Npad + a];
            v = d.v[slot * img + (size_t)c * d.Npad + a];
        } else {
            x = Xc[3 * (a - d.N) + c];
            v = d.vc[slot * 9 + 3 * (a - d.N) + c];
        }
        if (Xo) Xo[((size_t)p * rows + ao) * 3 + c] = x;
        if (vo) vo[((size_t)p * rows + ao) * 3 + c] = movable ? v : 0.0;
    }
}

// Checkpoint, second half: the generalized coordinates each image's neighbour list was built at (Xb, Xcb) and the
// staleness accounting {max |R~_i - R~_i(build)|^2 at the last K0, max |dR~_i|^2 of the last update, steps since
// the build, pending} -- what cfneb_set_state needs to replay the list builds and continue bit for bit.  pending is
// what host-side moves since the last K0 left for the next one: max |dR~_i|^2 of a path replacement / state import /
// re-parametrisation (dispmax_in), or -1 when the image's list must be rebuilt whatever moved (a new image, whose
// stored build coordinates mean nothing).
__global__ void export_list_state_kernel(Dev d, double *Xo, double *aux) {
    const int p = blockIdx.y;
    const int P = d.ctl->P;
    if (p >= P) return;
    const int slot = d.order[p];
    const int rows = d.N + 3;
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a == 0 && aux) {
        aux[4 * p + 0] = bits_nonneg(d.disptot[slot]);
        aux[4 * p + 1] = bits_nonneg(d.dispmax[slot]);
        aux[4 * p + 2] = (double)d.geom[slot].since;
        aux[4 * p + 3] = d.geom[slot].force_rebuild ? -1.0 : bits_nonneg(d.dispmax_in[slot]);
    }
    if (a >= rows || !Xo) return;
    const double *Xb = d.Xb + (size_t)slot * 3 * d.Npad;
    const int ao = a < d.N ? d.perm[a] : a;
    for (int c = 0; c < 3; ++c)
        Xo[((size_t)p * rows + ao) * 3 + c] = a < d.N ? Xb[(size_t)c * d.Npad + a] : d.Xcb[slot * 9 + 3 * (a - d.N) + c];
}

// Host-side moves (state import with tracking, re-parametrisation) record their largest atomic displacement in
// dispmax_in by atomicMax, which is right for the blocks of ONE move but not across moves: two moves with no K0
// between them can add up (triangle inequality) while the maximum only keeps the larger.  Run before such a move:
// an image that still carries an unconsumed displacement gets its list rebuilt by the next K0, whatever the sum is.
__global__ void pending_guard_kernel(Dev d, int p_first, int count) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int p = p_first + k;
    if (k >= count || p >= d.ctl->P) return;
    const int slot = d.order[p];
    if (d.dispmax_in[slot] != 0ull) d.geom[slot].force_rebuild = 1;
}

// Inverse of export_state_kernel: X (and v, if given) from the caller's layout into both coordinate buffers.
// track: the largest atomic displacement of each image from the stored coordinates goes into the staleness bound of
// its neighbour list (as cfneb_set_path does), so the lists are kept while the new state stays inside their skin.
__global__ void import_state_kernel(Dev d, const double *__restrict__ Xi, const double *__restrict__ vi, int track, int p_first,
                                    int count) {
    const int p = p_first + blockIdx.y;
    const int P = d.ctl->P;
    if ((int)blockIdx.y >= count || p >= P) return;
    const int slot = d.order[p];
    const int rows = d.N + 3;
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    const size_t img = (size_t)3 * d.Npad, buf = (size_t)d.S * img;
    const bool movable = p > 0 && p < P - 1;
    const int ai = a < d.N ? d.perm[a] : a;
    if (track) {  // all threads of the block take part in the reduction
        __shared__ double red[32];
        double d2 = 0.0;
        if (a < d.N) {
            const double *Xold = d.X + (size_t)d.ctl->cur * buf + slot * img;
            for (int c = 0; c < 3; ++c) {
                const double dx = Xi[((size_t)p * rows + ai) * 3 + c] - Xold[(size_t)c * d.Npad + a];
                d2 += dx * dx;
            }
            if (!(d2 == d2)) d2 = 1e300;
        }
        const double bm = block_max(d2, red);
        if (threadIdx.x == 0) atomicMax(d.dispmax_in + slot, nonneg_bits(bm));
    }
    if (a >= rows) return;
    for (int c = 0; c < 3; ++c) {
        const double x = Xi[((size_t)p * rows + ai) * 3 + c];
        const double v = (vi && movable) ? vi[((size_t)p * rows + ai) * 3 + c] : 0.0;
        if (a < d.N) {
            d.X[slot * img + (size_t)c * d.Npad + a] = x;
            d.X[buf + slot * img + (size_t)c * d.Npad + a] = x;
            if (vi) d.v[slot * img + (size_t)c * d.Npad + a] = v;
        } else {
            const int k = 3 * (a - d.N) + c;
            d.Xc[slot * 9 + k] = x;
            d.Xc[(size_t)d.S * 9 + slot * 9 + k] = x;
            if (vi) d.vc[slot * 9 + k] = v;
        }
    }
}

__global__ void import_aux_kernel(Dev d, const double *aux, int have_aux, int have_fire, double dt, double alpha, int n_pos,
                                  int first, unsigned long long steps) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (have_aux && p < d.ctl->P) {
        const int slot = d.order[p];
        d.disptot[slot] = nonneg_bits(aux[4 * p + 0]);
        d.dispmax[slot] = nonneg_bits(aux[4 * p + 1]);
        const double pending = aux[4 * p + 3];
        d.dispmax_in[slot] = pending > 0.0 ? nonneg_bits(pending) : 0ull;
        if (pending < 0.0) d.geom[slot].force_rebuild = 1;  // the replay built this list at X itself; K0 builds it again
        d.geom[slot].since = (int)aux[4 * p + 2];
    }
    if (p == 0 && have_fire) {
        Ctl *c = d.ctl;
        c->dt = dt;
        c->alpha = alpha;
        c->n_pos = n_pos;
        c->first = first;
        c->steps = steps;
    }
}

__global__ void export_forces_kernel(Dev d, double *Fo, double *Vo, double *Eo) {
    const int p = blockIdx.y;
    if (p >= d.ctl->P) return;
    const int slot = d.order[p];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < d.N && Fo) {
        const double *F = d.F + (size_t)slot * 3 * d.Npad;
        double *o = Fo + ((size_t)p * d.N + d.perm[i]) * 3;
        o[0] = F[i]; o[1] = F[d.Npad + i]; o[2] = F[2 * (size_t)d.Npad + i];
    }
    if (blockIdx.x == 0 && threadIdx.x < 9 && Vo) Vo[p * 9 + threadIdx.x] = d.V[slot * 9 + threadIdx.x];
    if (blockIdx.x == 0 && threadIdx.x == 0 && Eo) Eo[p] = d.E[slot];
}

void launch_update(const Dev &d, cudaStream_t st) {
    if (d.S < 3) return;
    dim3 grid(d.nblk_upd, d.S - 2);
    update_kernel<3><<<grid, kThreadsStream, 0, st>>>(d);
}

int update_blocks_per_sm() { return 3; }

void launch_materialize_fneb(const Dev &d, cudaStream_t st) {
    dim3 grid((d.N + 3 + 127) / 128, d.S);
    materialize_fneb_kernel<<<grid, 128, 0, st>>>(d);
}

void launch_materialize_gen_force(const Dev &d, cudaStream_t st) {
    dim3 grid((d.N + 3 + 127) / 128, d.S);
    materialize_gen_force_kernel<<<grid, 128, 0, st>>>(d);
}

void launch_export_dots(const Dev &d, double *dots_out, double *coef_out, cudaStream_t st) {
    export_dots_kernel<<<1, 256, 0, st>>>(d, dots_out, coef_out);
}

void launch_midpoint(const Dev &d, int sa, int sb, int sn, cudaStream_t st) {
    const size_t n = (size_t)3 * d.Npad;
    midpoint_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d, sa, sb, sn);
}

void launch_reset_fire(const Dev &d, cudaStream_t st) { reset_fire_kernel<<<592, 256, 0, st>>>(d); }

void launch_segment_lengths(const Dev &d, double *out_dev, cudaStream_t st) {
    segment_lengths_kernel<<<d.S - 1, 256, 0, st>>>(d, out_dev);
}

void launch_export_path(const Dev &d, double *pos_out, double *cells_out, double *E_out, cudaStream_t st) {
    dim3 grid(d.nblk_atom, d.S);
    export_path_kernel<<<grid, kThreadsAtom, 0, st>>>(d, pos_out, cells_out, E_out);
}

void launch_export_state(const Dev &d, double *X_out, double *v_out, cudaStream_t st) {
    dim3 grid((d.N + 3 + 127) / 128, d.S);
    export_state_kernel<<<grid, 128, 0, st>>>(d, X_out, v_out);
}

void launch_export_list_state(const Dev &d, double *Xl_out, double *aux_out, cudaStream_t st) {
    dim3 grid((d.N + 3 + 127) / 128, d.S);
    export_list_state_kernel<<<grid, 128, 0, st>>>(d, Xl_out, aux_out);
}

void launch_import_state(const Dev &d, const double *X_in, const double *v_in, int track, int p_first, int count,
                         cudaStream_t st) {
    if (count <= 0) return;
    if (track) launch_pending_guard(d, p_first, count, st);
    dim3 grid((d.N + 3 + 127) / 128, count);
    import_state_kernel<<<grid, 128, 0, st>>>(d, X_in, v_in, track, p_first, count);
}

void launch_pending_guard(const Dev &d, int p_first, int count, cudaStream_t st) {
    if (count <= 0) return;
    pending_guard_kernel<<<(count + 127) / 128, 128, 0, st>>>(d, p_first, count);
}

void launch_import_aux(const Dev &d, const double *aux_in, int have_aux, int have_fire, double dt, double alpha, int n_pos,
                       int first, unsigned long long steps, cudaStream_t st) {
    import_aux_kernel<<<(d.S + 127) / 128, 128, 0, st>>>(d, aux_in, have_aux, have_fire, dt, alpha, n_pos, first, steps);
}

void launch_export_forces(const Dev &d, double *F_out, double *V_out, double *E_out, cudaStream_t st) {
    dim3 grid(d.nblk_atom, d.S);
    export_forces_kernel<<<grid, kThreadsAtom, 0, st>>>(d, F_out, V_out, E_out);
}

}  // namespace cfn

// kernels_cell.cu -- cell filter geometry: input mapping (O0, Eq. 10/15), cell map D = sqrt(B) (O1, P:110,
// P:119-124, reading A8), Cartesian positions R = R~ D, and the device-side decision to rebuild neighbour lists.
#include "cfneb_internal.cuh"

namespace cfn {

// Symmetric positive-definite square root of a symmetric 3x3 matrix by cyclic Jacobi (fp64, to convergence).
// Returns false if an eigenvalue is not positive.
__device__ bool sqrt_spd3(const double *Bin, double *S) {
    double A[9], U[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1};
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) A[3 * i + j] = 0.5 * (Bin[3 * i + j] + Bin[3 * j + i]);
    for (int sweep = 0; sweep < 60; ++sweep) {
        double off = A[1] * A[1] + A[2] * A[2] + A[5] * A[5];
        double dia = A[0] * A[0] + A[4] * A[4] + A[8] * A[8];
        if (off <= 1e-33 * (dia + 2.0 * off) || off == 0.0) break;
        for (int pq = 0; pq < 3; ++pq) {
            const int p = (pq == 2) ? 1 : 0, q = (pq == 0) ? 1 : 2;
            double apq = A[3 * p + q];
            if (apq == 0.0) continue;
            double theta = (A[3 * q + q] - A[3 * p + p]) / (2.0 * apq);
            double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
            double c = 1.0 / sqrt(t * t + 1.0), s = t * c;
            for (int k = 0; k < 3; ++k) {  // A <- A J (columns p, q)
                double akp = A[3 * k + p], akq = A[3 * k + q];
                A[3 * k + p] = c * akp - s * akq;
                A[3 * k + q] = s * akp + c * akq;
            }
            for (int k = 0; k < 3; ++k) {  // A <- J^T A (rows p, q)
                double apk = A[3 * p + k], aqk = A[3 * q + k];
                A[3 * p + k] = c * apk - s * aqk;
                A[3 * q + k] = s * apk + c * aqk;
            }
            for (int k = 0; k < 3; ++k) {  // U <- U J
                double ukp = U[3 * k + p], ukq = U[3 * k + q];
                U[3 * k + p] = c * ukp - s * ukq;
                U[3 * k + q] = s * ukp + c * ukq;
            }
        }
    }
    double w0 = A[0], w1 = A[4], w2 = A[8];
    if (!(w0 > 0.0) || !(w1 > 0.0) || !(w2 > 0.0)) return false;
    double r0 = sqrt(w0), r1 = sqrt(w1), r2 = sqrt(w2);
    for (int i = 0; i < 3; ++i)
        for (int j = i; j < 3; ++j) {
            double x = U[3 * i] * r0 * U[3 * j] + U[3 * i + 1] * r1 * U[3 * j + 1] + U[3 * i + 2] * r2 * U[3 * j + 2];
            S[3 * i + j] = x;
            S[3 * j + i] = x;
        }
    return true;
}

// Smallest eigenvalue of a symmetric 3x3 matrix (cyclic Jacobi to convergence).
__device__ double min_eig_sym3(const double *Cin) {
    double A[9];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) A[3 * i + j] = 0.5 * (Cin[3 * i + j] + Cin[3 * j + i]);
    for (int sweep = 0; sweep < 60; ++sweep) {
        const double off = A[1] * A[1] + A[2] * A[2] + A[5] * A[5];
        const double dia = A[0] * A[0] + A[4] * A[4] + A[8] * A[8];
        if (off <= 1e-33 * (dia + 2.0 * off) || off == 0.0) break;
        for (int pq = 0; pq < 3; ++pq) {
            const int p = (pq == 2) ? 1 : 0, q = (pq == 0) ? 1 : 2;
            const double apq = A[3 * p + q];
            if (apq == 0.0) continue;
            const double theta = (A[3 * q + q] - A[3 * p + p]) / (2.0 * apq);
            const double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
            const double c = 1.0 / sqrt(t * t + 1.0), s = t * c;
            for (int k = 0; k < 3; ++k) {
                const double akp = A[3 * k + p], akq = A[3 * k + q];
                A[3 * k + p] = c * akp - s * akq;
                A[3 * k + q] = s * akp + c * akq;
            }
            for (int k = 0; k < 3; ++k) {
                const double apk = A[3 * p + k], aqk = A[3 * q + k];
                A[3 * p + k] = c * apk - s * aqk;
                A[3 * q + k] = s * apk + c * aqk;
            }
        }
    }
    return fmin(A[0], fmin(A[4], A[8]));
}

// Upper bound of the spectral norm: ||m||_2 <= sqrt(||m||_1 ||m||_inf) (tight for the near-identity,
// symmetric D of CELL_B, unlike the Frobenius norm).
__device__ inline double norm2_bound(const double *m) {
    double r = 0.0, c = 0.0;
    for (int i = 0; i < 3; ++i) {
        r = fmax(r, fabs(m[3 * i]) + fabs(m[3 * i + 1]) + fabs(m[3 * i + 2]));
        c = fmax(c, fabs(m[i]) + fabs(m[3 + i]) + fabs(m[6 + i]));
    }
    return sqrt(r * c);
}

// O0: one block column per image; pos [count][N][3] Cartesian, cells [count][9] are images p_first.. of the path.
// Writes R~ = R D^-1 into both X buffers and lam*B (or lam*D) into both Xc buffers of slot = order[p].
__global__ void input_map_kernel(Dev d, const double *__restrict__ pos, const double *__restrict__ cells, int p_first,
                                 int count, int track) {
    const int p = blockIdx.y;  // local index into pos / cells
    if (p >= count) return;
    const int slot = d.order[p_first + p];
    double D[9], Dinv[9];
    mul3(d.h0inv, cells + 9 * p, D);  // D = h0^-1 h
    inv3(D, Dinv);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const size_t img = (size_t)3 * d.Npad, buf = (size_t)d.S * img;
    double d2 = 0.0;
    if (i < d.N) {
        const double *r = pos + ((size_t)p * d.N + d.perm[i]) * 3;  // caller's order -> spatial storage order
        const double *Xold = d.X + (size_t)d.ctl->cur * buf + slot * img;
        for (int c = 0; c < 3; ++c) {
            double x = r[0] * Dinv[c] + r[1] * Dinv[3 + c] + r[2] * Dinv[6 + c];  // R~ = R D^-1 (Eq. 10)
            if (track) { const double dx = x - Xold[(size_t)c * d.Npad + i]; d2 += dx * dx; }
            d.X[slot * img + (size_t)c * d.Npad + i] = x;
            d.X[buf + slot * img + (size_t)c * d.Npad + i] = x;
        }
    }
    if (track) {  // the neighbour list of this slot stays valid if the new path is within the skin of the old one
        __shared__ double red[32];
        if (!(d2 == d2)) d2 = 1e300;  // NaN input: force a rebuild (and the NaN check of the evaluation)
        const double bm = block_max(d2, red);
        if (threadIdx.x == 0) atomicMax(d.dispmax_in + slot, nonneg_bits(bm));
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        double C[9];
        if (d.cell_mode == CFNEB_CELL_D) for (int k = 0; k < 9; ++k) C[k] = D[k];
        else mul3_abt(D, D, C);  // B = D D^T (Eq. 15)
        for (int k = 0; k < 9; ++k) {
            d.Xc[slot * 9 + k] = d.lam * C[k];
            d.Xc[(size_t)d.S * 9 + slot * 9 + k] = d.lam * C[k];
        }
        if (!(det3(cells + 9 * p) != 0.0)) set_error(d.ctl, CFNEB_ECELL);
    }
}

// Interior images linear in generalized coordinates between the endpoints (create without an explicit path).
__global__ void interpolate_kernel(Dev d, int P) {
    const int p = blockIdx.y + 1;
    if (p >= P - 1) return;
    const int s0 = d.order[0], s1 = d.order[P - 1], slot = d.order[p];
    const double t = (double)p / (double)(P - 1);
    const size_t img = (size_t)3 * d.Npad, buf = (size_t)d.S * img;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < 3 * d.Npad) {
        double a = d.X[s0 * img + i], b = d.X[s1 * img + i];
        double x = a + t * (b - a);
        d.X[slot * img + i] = x;
        d.X[buf + slot * img + i] = x;
    }
    if (blockIdx.x == 0 && threadIdx.x < 9) {
        double a = d.Xc[s0 * 9 + threadIdx.x], b = d.Xc[s1 * 9 + threadIdx.x];
        double x = a + t * (b - a);
        d.Xc[slot * 9 + threadIdx.x] = x;
        d.Xc[(size_t)d.S * 9 + slot * 9 + threadIdx.x] = x;
    }
}

// K0: per image, D = sqrt(B), D^-1, h = h0 D, Omega; staleness bound of the neighbour list and the
// rebuild decision; zeroes the bin counters of images that rebuild.
__global__ void cell_prep_kernel(Dev d, int p_lo, int mode) {
    const int P = d.ctl->P;
    int p;
    if (!image_of(blockIdx.x, p_lo, P, p)) return;
    const int slot = d.order[p];
    Geom *g = d.geom + slot;
    __shared__ int s_rebuild, s_nbins;
    if (threadIdx.x == 0) {
        const double *xc = d.Xc + (size_t)d.ctl->cur * d.S * 9 + slot * 9;
        double C[9], D[9], Dinv[9], h[9];
        for (int k = 0; k < 9; ++k) C[k] = xc[k] / d.lam;
        bool ok = true;
        if (d.cell_mode == CFNEB_CELL_D) for (int k = 0; k < 9; ++k) D[k] = C[k];
        else ok = sqrt_spd3(C, D);
        int rebuild = 0, nbins = 0;
        if (!ok) set_error(d.ctl, CFNEB_ECELL);
        else {
            mul3(d.h0, D, h);
            double vol = det3(h);
            if (!(fabs(vol) > 0.0) || !isfinite(vol)) { set_error(d.ctl, CFNEB_ECELL); ok = false; }
            if (ok) {
                inv3(D, Dinv);
                if (mode == MODE_STEP) {
                    // How much closer than at the build any pair can be now.  With r = (dR~ + n h0) D, M = Db^-1 D and
                    // d_i = R~_i - R~_i(build):   |r| >= sigma_min(M) |r_build| - 2 max_i |d_i| ||D||,   so a pair that
                    // was outside r_list cannot be inside r_cut while
                    //   acc = 2 max_i |d_i| ||D|| + r_list (1 - sigma_min(M))_+  <=  skin,
                    // and a list entry built at r_build >= r_cut + acc is still outside r_cut (tail buckets of K2).
                    // Only compression brings pairs in: an expanding or shearing cell costs nothing beyond
                    // 1 - sigma_min (the norm ||D - Db|| used before was 2-3 x larger on the Bain band).
                    // max_i |d_i| was measured exactly by positions_kernel at the last K0 (disptot); what moved since --
                    // the last update (dispmax), a path replacement (dispmax_in) -- is added by the triangle inequality.
                    // Not cumulative: FIRE makes atoms oscillate, and the sum of per-step maxima that this replaced was
                    // 6-16 times the true displacement at c4.
                    const double dmax = sqrt(bits_nonneg(d.disptot[slot])) + sqrt(bits_nonneg(d.dispmax[slot])) +
                                        sqrt(bits_nonneg(d.dispmax_in[slot]));
                    double M[9], C[9];
                    mul3(g->Dbinv, D, M);
                    mul3_atb(M, M, C);  // M^T M
                    const double lmin = min_eig_sym3(C);
                    const double smin = lmin > 0.0 ? sqrt(lmin) : 0.0;
                    const double shrink = 1.0 - smin;  // + a rounding allowance of the 3x3 arithmetic when it counts
                    double acc = 2.0 * dmax * norm2_bound(D) + d.r_list * (shrink > 0.0 ? shrink * (1.0 + 1e-12) + 1e-14 : 0.0);
                    d.dispmax[slot] = 0ull;
                    d.dispmax_in[slot] = 0ull;
                    d.disptot[slot] = 0ull;  // positions_kernel of this step measures it again
                    rebuild = g->force_rebuild || !(acc <= d.skin) || (d.rebuild_every > 0 && g->since + 1 >= d.rebuild_every);
                    if (rebuild) {
                        acc = 0.0;
                        g->since = 0;
                        g->force_rebuild = 0;
                        for (int k = 0; k < 9; ++k) { g->Dbinv[k] = Dinv[k]; d.Xcb[slot * 9 + k] = xc[k]; }
                    } else {
                        g->since += 1;
                    }
                    g->acc = acc;
                }
                for (int k = 0; k < 9; ++k) { g->D[k] = D[k]; g->Dinv[k] = Dinv[k]; g->h[k] = h[k]; }
                g->vol = vol;
                if (rebuild) {
                    nbins = 1;
                    for (int a = 0; a < 3; ++a) {
                        const double *b = h + 3 * ((a + 1) % 3), *c = h + 3 * ((a + 2) % 3);
                        double cx = b[1] * c[2] - b[2] * c[1], cy = b[2] * c[0] - b[0] * c[2], cz = b[0] * c[1] - b[1] * c[0];
                        double w = fabs(vol) / sqrt(cx * cx + cy * cy + cz * cz);  // perpendicular width
                        int nb = (int)floor(w / d.r_list);
                        if (nb >= 3) { g->nb[a] = min(nb, max(d.nb_cap[a], 3)); g->reach[a] = 1; }
                        else { g->nb[a] = 1; g->reach[a] = (int)ceil(d.r_list / w); }
                        nbins *= g->nb[a];
                    }
                    if (nbins > d.nbins_max) { set_error(d.ctl, CFNEB_ECELL); rebuild = 0; }
                    else atomicAdd(&d.ctl->rebuilds, 1ull);
                }
            }
        }
        if (mode == MODE_STEP) g->rebuild = rebuild;
        s_rebuild = (mode == MODE_STEP) ? rebuild : 0;
        s_nbins = nbins;
    }
    __syncthreads();
    if (s_rebuild) {
        int *bc = d.bin_count + (size_t)slot * (d.nbins_max + 1);
        for (int b = threadIdx.x; b <= s_nbins; b += blockDim.x) bc[b] = 0;
    }
}

// Cartesian positions Rc = R~ D (one 32-byte sector per atom); when the slot rebuilds its list also
// wrapped fractional coordinates s = R~ h0^-1 (image independent, Eq. 10), bin index and bin population.
__global__ void __launch_bounds__(kThreadsAtom) positions_kernel(Dev d, int p_lo, int mode) {
    int p;
    if (!image_of(blockIdx.y, p_lo, d.ctl->P, p)) return;
    const int slot = d.order[p];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const Geom *g = d.geom + slot;
    if (mode == MODE_STEP && !g->rebuild) {
        // exact displacement of every atom from the coordinates its list was built at (K0 of the next step adds
        // what the update in between moves); all threads of the block take part in the reduction
        __shared__ double red[32];
        double d2 = 0.0;
        if (i < d.N) {
            const double *Xc = d.X + ((size_t)d.ctl->cur * d.S + slot) * 3 * d.Npad;
            const double *Xb = d.Xb + (size_t)slot * 3 * d.Npad;
            const double ax = Xc[i] - Xb[i], ay = Xc[d.Npad + i] - Xb[d.Npad + i],
                         az = Xc[2 * (size_t)d.Npad + i] - Xb[2 * (size_t)d.Npad + i];
            d2 = ax * ax + ay * ay + az * az;
            if (!(d2 == d2)) d2 = 1e300;
        }
        const double bm = block_max(d2, red);
        if (threadIdx.x == 0) atomicMax(d.disptot + slot, nonneg_bits(bm));
    }
    if (i >= d.N) return;
    const double *X = d.X + ((size_t)d.ctl->cur * d.S + slot) * 3 * d.Npad;
    const double x = X[i], y = X[d.Npad + i], z = X[2 * (size_t)d.Npad + i];
    double4 r;
    r.x = x * g->D[0] + y * g->D[3] + z * g->D[6];
    r.y = x * g->D[1] + y * g->D[4] + z * g->D[7];
    r.z = x * g->D[2] + y * g->D[5] + z * g->D[8];
    r.w = d.types ? (double)d.types[i] : 0.0;  // NEP: the atom type rides in the sector (FS: F'(rho), K2a)
    d.Rc[(size_t)slot * d.Npad + i] = r;
    if (mode == MODE_STEP && g->rebuild) {  // the list is built from these coordinates
        double *Xb = d.Xb + (size_t)slot * 3 * d.Npad;
        Xb[i] = x; Xb[d.Npad + i] = y; Xb[2 * (size_t)d.Npad + i] = z;
    }
    if (mode == MODE_STEP && g->rebuild) {
        double s[3], sw[3];
        int fl[3], b[3];
        s[0] = x * d.h0inv[0] + y * d.h0inv[3] + z * d.h0inv[6];
        s[1] = x * d.h0inv[1] + y * d.h0inv[4] + z * d.h0inv[7];
        s[2] = x * d.h0inv[2] + y * d.h0inv[5] + z * d.h0inv[8];
        bool bad = false;
        for (int a = 0; a < 3; ++a) {
            double f = floor(s[a]);
            sw[a] = s[a] - f;
            fl[a] = (int)f;
            if (!(fabs(f) < 500.0)) { bad = true; fl[a] = 0; }
            b[a] = (int)(sw[a] * g->nb[a]);
            if (b[a] >= g->nb[a]) b[a] = g->nb[a] - 1;
            if (b[a] < 0) b[a] = 0;
        }
        if (bad) set_error(d.ctl, CFNEB_ENAN);
        const int bin = (b[0] * g->nb[1] + b[1]) * g->nb[2] + b[2];
        unsigned long long packed = (unsigned long long)(fl[0] + 512) | ((unsigned long long)(fl[1] + 512) << 10) |
                                    ((unsigned long long)(fl[2] + 512) << 20);
        double4 w4;
        w4.x = sw[0]; w4.y = sw[1]; w4.z = sw[2];
        w4.w = __longlong_as_double((long long)packed);
        d.Sw[(size_t)slot * d.Npad + i] = w4;
        d.atom_bin[(size_t)slot * d.Npad + i] = bin;
        atomicAdd(d.bin_count + (size_t)slot * (d.nbins_max + 1) + bin, 1);
    }
}

void launch_input_map(const Dev &d, const double *pos_dev, const double *cells_dev, int p_first, int count, int track,
                      cudaStream_t st) {
    if (count <= 0) return;
    dim3 grid(d.nblk_atom, count);
    input_map_kernel<<<grid, kThreadsAtom, 0, st>>>(d, pos_dev, cells_dev, p_first, count, track);
}

void launch_interpolate(const Dev &d, int P, cudaStream_t st) {
    if (P < 3) return;
    dim3 grid((3 * d.Npad + 255) / 256, P - 2);
    interpolate_kernel<<<grid, 256, 0, st>>>(d, P);
}

void launch_cell_prep(const Dev &d, int p_lo, int mode, cudaStream_t st) {
    const int nimg = images_in_grid(d.S, p_lo);
    cell_prep_kernel<<<nimg, 128, 0, st>>>(d, p_lo, mode);
    dim3 grid(d.nblk_atom, nimg);
    positions_kernel<<<grid, kThreadsAtom, 0, st>>>(d, p_lo, mode);
}

}  // namespace cfn

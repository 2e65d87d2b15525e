// cfneb_internal.cuh -- device-side layout and launch wrappers shared by the CUDA translation units.
// (Product code: shares nothing with oracle/.)
//
// HBM layout (fp64 SoA, one "slot" per image; path position p -> slot through the order table, so
// insertion / deletion never moves atom data).  Atoms are stored in a spatial (Morton) order fixed at create
// -- consecutive threads own neighbouring atoms, so the position gathers of a block stay inside L1 -- and
// `perm` maps back to the caller's order at the boundary (input map, exports, parity hooks):
//   X    [2][S][3][Npad]   R~ of Eq. 10, double-buffered (K6 reads X_{p-1}, X_p, X_{p+1} of buffer src,
//                          writes buffer dst); rows padded with zeros to Npad (multiple of 32)
//   v, F [S][3][Npad]      FIRE velocity, Cartesian force (Eq. 5)
//   Rc   [S][Npad] double4 Cartesian position R = R~ D packed as one 32-byte sector per atom;
//                          .w carries F'(rho_i) between the two Finnis-Sinclair passes
//   Xc   [2][S][9], vc [S][9]   cell block lam*B (Eq. 17) and its velocity
//   nbr_list [S][cap][Npad] uint32: j | shift code << 23, k-major so that a warp reads 128 contiguous bytes
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/cfneb.h"

namespace cfn {

constexpr int kThreadsAtom = 128;      // neighbour / position / many-body kernels: 1 atom per thread
#ifndef CFNEB_PAIR_THREADS
#define CFNEB_PAIR_THREADS 128
#endif
constexpr int kThreadsPair = CFNEB_PAIR_THREADS;  // pair-potential K2 kernels (density, force): 1 atom per thread
constexpr int kThreadsStream = 256;    // K4 / K6: 2 atoms per thread (double2)
constexpr int kAtomsPerStreamBlock = kThreadsStream * 2;
constexpr int kHistLen = CFNEB_HISTORY_LEN;  // iterations kept in the per-step record (ring), cfneb_get_history
constexpr int kHistFields = 8;          // steps after the iteration, |f|max^2, barrier, p*, dt, alpha, P, rebuilds
constexpr int kNDots = 10;             // pp, mm, pm, Gp, Gm, GG, Gv, pv, mv, vv
constexpr int kNForcePart = 10;        // E pair, Vxx, Vyy, Vzz, Vxy, Vxz, Vyz, E site (embedding / many-body), low words of [0], [7]
constexpr uint32_t kIdxMask = 0x7FFFFFu;
constexpr int kShiftBits = 23;
constexpr uint32_t kCodeCenter = 4u | (4u << 3) | (4u << 6);
constexpr int kMaxAtoms = 1 << 23;
constexpr int kDnWeights = 8 * 16 + 2 * 8;  // CFNEB_POT_DNN: H <= 8, D <= 16
constexpr int kInnerBuckets = 56;      // radial buckets of the list sort: uniform in r^2 on [0, r_cut^2)
constexpr int kTailBuckets = 8;        // ... and on [r_cut^2, r_list^2)
constexpr int kQueueSlack = 32;        // rows of the K1 candidate queue beyond the list capacity (prefilter margin)
constexpr int kEdgeRows = 12;          // inner bucket edges from Dev::edge_b0 on whose list offsets are kept (Dev::nbr_edge)

enum { DOT_PP = 0, DOT_MM, DOT_PM, DOT_GP, DOT_GM, DOT_GG, DOT_GV, DOT_PV, DOT_MV, DOT_VV };

// Device-resident control block: everything the graph needs to run step after step with no host round trip.
struct Ctl {
    int P;            // current number of images
    int cur;          // X buffer holding the latest coordinates
    int src, dst;     // set by K5 for K6 of the same step
    int error;        // sticky CFNEB_E* code
    int first;        // FIRE: skip the power test on the first step after a (re)start (A2)
    int n_pos;
    int pstar;        // climbing image (path position) of the last step
    int max_nbr_seen;
    int pad0;
    unsigned long long steps;
    unsigned long long rebuilds;
    double dt, alpha;
    double cv, cf, sdt;   // K6: v_new = cv v + cf f ; X_new = X + sdt v_new
    unsigned long long fmax_bits;  // max row norm^2 of f as ordered bits (atomicMax target)
    double barrier, path_length;
    // device-side adaptive control (kernels_adapt.cu)
    int n_free;                   // free-slot stack height (free_stack[0 .. n_free-1], top last)
    int ins_a, ins_b, ins_new;    // slots of a pending midpoint insertion, ins_new < 0: none
    int changed;                  // the last control step changed the band (FIRE restart pending)
    int n_inserted, n_deleted;    // totals since create
    int n_rebuild;                // images whose neighbour list is rebuilt this step (rebuild_slots[0 .. n_rebuild-1])
};

// FIRE state of one endpoint during cfneb_relax_endpoints (kernels_relax.cu); device resident.
struct RelaxState {
    double dt, alpha;
    double cv, cf, sdt;   // v_new = cv v + cf G ; X_new = X + sdt v_new
    double fmax, E;       // max row norm of G and energy at the last evaluation
    int n_pos, first, frozen, steps;
};

// Per-slot geometry written by K0.
struct Geom {
    double D[9], Dinv[9], h[9];
    double Dbinv[9];   // inverse of D at the time the neighbour list of this slot was built
    double vol;
    double acc;        // bound on the change of any pair distance since the last list build (K0, every step)
    int nb[3];         // bins per axis (>= 3: adjacent-bin stencil; 1: explicit periodic shifts)
    int reach[3];      // stencil half-width per axis
    int rebuild;       // this step rebuilds the list of this slot
    int force_rebuild; // set by host paths (create / insert / set_path)
    int since;         // steps since last build
    int pad;
};

struct Dev {
    int N, Npad, S, cap;      // cap: list rows per atom = max_neighbors rounded up to even
    int cap_user;             // max_neighbors as given: the overflow threshold and the row length of cfneb_get_neighbors
    int potential, cell_mode, climb, fire_nmin, rebuild_every;
    int nblk_atom, nblk_stream, nbins_max;
    int nblk_force;           // blocks per image of the K2 kernels that write part_force (pair kernels: kThreadsPair atoms each)
    int n_sm;                 // multiprocessors of the device
    int n_search_blocks;      // grid of neighbor_search_kernel (resident blocks: n_sm x blocks per SM)
    int nblk_red, nblk_upd;   // K4 / K6: blocks per image, each striding over the image's nblk_stream tiles
    int nb_cap[3];
    double pot[12];
    double potc[24];          // derived potential constants (kernels_force.cu: prepare_potential)
    double k_spring, lam;
    double pressure;          // external hydrostatic pressure (A25): E <- U + p Omega, V <- V - p Omega I in finalize_kernel
    double dt0, dtmax, maxstep, finc, fdec, astart, fa;
    double skin, r_cut, r_list;
    double h0[9], h0inv[9];
    Ctl *ctl;
    int *order;               // [S] path position -> slot
    int *free_stack;          // [S] unused slots (device-side adaptive control)
    double *hist;             // [kHistLen][kHistFields] per-iteration record written by K5 (row = iteration index mod kHistLen)
    double *seglen;           // [2 S] segment lengths of the last control step; second half: running arc length
    int *plan_q;              // [S] re-parametrisation: image p moves onto segment plan_q[p] ...
    double *plan_t;           // [S] ... at the fraction plan_t[p] (kernels_adapt.cu)
    int *perm;                // [Npad] internal atom index -> caller's atom index (spatial order, see api.cu)
    Geom *geom;               // [S]
    double *X, *v, *F;        // see header comment
    double *fneb;             // parity-hook scratch [S][(N+3)*3], external row-major layout
    double4 *Rc;
    double4 *Sw;              // [S][Npad] wrapped fractional coordinates + packed floors, for the list build
    double4 *binned;          // [S][Npad] Sw in bin order, .w = packed (atom index, floors)
    float4 *binned_c;         // [S][Npad] fp32 Cartesian wrapped positions in bin order (prefilter of the search)
    double *Xc, *vc;
    double *E, *V, *Gc;       // [S], [S][9], [S][9]
    double *dots, *coef;      // [S][10], [S][4]
    double *part_force;       // [S][nblk_force][kNForcePart]
    RelaxState *relax;        // [2]
    double *part_relax;       // [2][nblk_stream][4]
    double *part_dots;        // [S][nblk_stream][10]  (the first nblk_red rows of an image are used)
    unsigned long long *dispmax;  // [S] max |dR~_i|^2 of the last update, as ordered bits
    unsigned long long *disptot;  // [S] max |R~_i - R~_i(build)|^2 at the last K0, as ordered bits
    double *Xb;                   // [S][3][Npad] R~ at the last list build of each slot
    double *Xcb;                  // [S][9] cell rows lam B (lam D) at the last list build (checkpoint: the build is replayed)
    unsigned long long *dispmax_in;  // [S] max |dR~_i|^2 of a path replacement (cfneb_set_path) since the last K0
    int *nbr_count;           // [S][Npad]
    uint32_t *nbr_list;       // [S][cap][Npad]  Verlet list (r < r_cut + skin), sorted by distance at build, rebuilt when stale
    unsigned short *nbr_tail; // [S][kTailBuckets][Npad] number of entries below tail bucket t (list sorted by bucket)
    unsigned short *nbr_edge; // [S][kEdgeRows][Npad] number of entries below inner bucket edge_b0 + q (NEP: the rows
                              // that can lie inside the angular cut-off; nullptr for the other potentials)
    int edge_b0;              // first inner bucket edge kept: the last one at or below the inner radius (NEP: rc_a)
    double *dn_w;               // [kDnWeights] W0[H][D], b0[H], W1[H] of CFNEB_POT_DNN; CFNEB_POT_NEP: see kernels_nep.cu
    int *types;                 // [Npad] atom types in storage order (CFNEB_POT_NEP)
    double *nep_q;              // [S][8][Npad] radial descriptors q_n (nep_radial_desc_kernel -> quad kernel)
    double *nep_w;              // [S][Npad][n_types][nep_kr_pad] w_i[J][k] = sum_n dU_i/dq_n cR[I][J][n][k] (quad kernel -> nep_radial_pair_kernel)
    int nep_kr_pad;             // k_r rounded up to 4, 8 or 12
    double *nep_S;              // [S][n_a][35][Npad] moments of the angular channels between the two walks (CFNEB_POT_NEP)
    unsigned short *nbr_mirror; // [S][cap][Npad] row of the mirror entry (j; i, -n) of each entry (many-body potentials only)
    double *part;             // [S][cap][3][Npad] partial forces p^ij = dU_i/dr^ij per list entry (many-body potentials only)
    int *rebuild_slots;       // [S] compact list of the slots that rebuild this step (K1)
    unsigned char *scr_bkt;   // [n_search_blocks][cap][128] r^2 bucket of each unsorted entry
    uint32_t *scr_queue;      // [n_search_blocks][cap + kQueueSlack][128] candidates that passed the fp32 prefilter, per atom;
                              // rewritten in place by the drain as the unsorted column of the block's current work item
    int *bin_count;           // [S][nbins_max + 1]  (counts, then exclusive starts)
    int *bin_cursor;          // [S][nbins_max]
    int *bin_members;         // [S][Npad]
    int *atom_bin;            // [S][Npad]
    void *scratch;            // staging for host transfers / hooks
    size_t scratch_bytes;
};

// ---- small 3x3 helpers, row-major ----
__host__ __device__ inline double det3(const double *m) {
    return m[0] * (m[4] * m[8] - m[5] * m[7]) - m[1] * (m[3] * m[8] - m[5] * m[6]) + m[2] * (m[3] * m[7] - m[4] * m[6]);
}
__host__ __device__ inline void inv3(const double *m, double *o) {
    double id = 1.0 / det3(m);
    o[0] = (m[4] * m[8] - m[5] * m[7]) * id; o[1] = (m[2] * m[7] - m[1] * m[8]) * id; o[2] = (m[1] * m[5] - m[2] * m[4]) * id;
    o[3] = (m[5] * m[6] - m[3] * m[8]) * id; o[4] = (m[0] * m[8] - m[2] * m[6]) * id; o[5] = (m[2] * m[3] - m[0] * m[5]) * id;
    o[6] = (m[3] * m[7] - m[4] * m[6]) * id; o[7] = (m[1] * m[6] - m[0] * m[7]) * id; o[8] = (m[0] * m[4] - m[1] * m[3]) * id;
}
__host__ __device__ inline void mul3(const double *a, const double *b, double *c) {  // c = a b
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) c[3 * i + j] = a[3 * i] * b[j] + a[3 * i + 1] * b[3 + j] + a[3 * i + 2] * b[6 + j];
}
__host__ __device__ inline void mul3_abt(const double *a, const double *b, double *c) {  // c = a b^T
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) c[3 * i + j] = a[3 * i] * b[3 * j] + a[3 * i + 1] * b[3 * j + 1] + a[3 * i + 2] * b[3 * j + 2];
}
__host__ __device__ inline void mul3_atb(const double *a, const double *b, double *c) {  // c = a^T b
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) c[3 * i + j] = a[i] * b[j] + a[3 + i] * b[3 + j] + a[6 + i] * b[6 + j];
}

// launch modes
enum { MODE_STEP = 0, MODE_GEOMETRY_ONLY = 1 };

// Image selection of the per-image kernels: p_lo = 1 the movable images 1..P-2, p_lo = 0 all images,
// p_lo = kEndpointsOnly the two endpoints (endpoint relaxation), p_lo = image_block(first, count) the movable images
// among `count` consecutive path positions from `first` (cfneb_step_hosted: image blocks are evaluated while later
// blocks are still on their way from the host).  y = the block's image coordinate.
constexpr int kEndpointsOnly = -1;
__host__ __device__ inline int image_block(int first, int count) { return -2 - (first | (count << 12)); }  // first, count < 4096
__host__ __device__ inline bool image_of(int y, int p_lo, int P, int &p) {
    if (p_lo == kEndpointsOnly) { p = y ? P - 1 : 0; return y < 2; }
    if (p_lo < kEndpointsOnly) {
        const int code = -2 - p_lo;
        p = (code & 4095) + y;
        return y < (code >> 12) && p >= 1 && p <= P - 2;
    }
    p = y + p_lo;
    return p <= P - 1 - p_lo;
}
__host__ __device__ inline int images_in_grid(int S, int p_lo) {
    return p_lo == kEndpointsOnly ? 2 : p_lo < kEndpointsOnly ? ((-2 - p_lo) >> 12) : S - 2 * p_lo;
}

// ---- launch wrappers (each enqueues on `st`; p_lo = 1: movable images, 0: all images) ----
void launch_input_map(const Dev &d, const double *pos_dev, const double *cells_dev, int p_first, int count, int track,
                      cudaStream_t st);  // track = 1: record the displacement against the stored coordinates
void launch_interpolate(const Dev &d, int P, cudaStream_t st);
void launch_cell_prep(const Dev &d, int p_lo, int mode, cudaStream_t st);                 // K0 + positions
void launch_neighbor_build(const Dev &d, int p_lo, cudaStream_t st);                      // K1
int search_blocks_per_sm();
void prepare_potential(Dev &d);  // fills Dev::potc from pot / r_cut (host)
void launch_force(const Dev &d, int p_lo, cudaStream_t st);
void launch_mirror_sw(const Dev &d, int p_lo, cudaStream_t st);                          // mirror rows after a list build
void launch_force_dn(const Dev &d, int p_lo, cudaStream_t st);                            // K2, descriptor network (kernels_dn.cu)
void launch_force_nep(const Dev &d, int p_lo, cudaStream_t st);                           // K2, NEP-shaped potential (kernels_nep.cu)
int nep_weight_count(const double *pot);
int nep_kr_padded(const double *pot);
void nep_fill_weights(const double *pot, double *w);  // host: the SplitMix64 weight stream of include/cfneb.h
void launch_pair_forces_manybody(const Dev &d, int p_lo, cudaStream_t st);                // pass 2 of both (kernels_sw.cu)
void launch_force_sw(const Dev &d, int p_lo, cudaStream_t st);                            // K2, Stillinger-Weber (kernels_sw.cu)                               // K2
void launch_reduce(const Dev &d, cudaStream_t st);                                        // K4 (atom rows)
void plan_stream_grids(Dev &d);  // nblk_red / nblk_upd from the SM count and the kernels' occupancy
void launch_finalize(const Dev &d, int p_lo, cudaStream_t st);                            // K4 second stage
void launch_scalar(const Dev &d, int dry, cudaStream_t st);                               // K5
void launch_update(const Dev &d, cudaStream_t st);                                        // K6
void launch_materialize_fneb(const Dev &d, cudaStream_t st);                              // parity hook
void launch_midpoint(const Dev &d, int slot_a, int slot_b, int slot_new, cudaStream_t st);  // K7
void launch_reset_fire(const Dev &d, cudaStream_t st);
void launch_adapt_device(const Dev &d, double d_insert, double d_delete, cudaStream_t st);  // O9 on the device
void launch_reparametrize(const Dev &d, int hold_climbing, cudaStream_t st);                // equal arc length (A27)
void launch_relax_init(const Dev &d, cudaStream_t st);                                    // endpoint relaxation
void launch_relax_step(const Dev &d, double fmax_tol, cudaStream_t st);
void launch_segment_lengths(const Dev &d, double *out_dev, cudaStream_t st);
cudaError_t prepare_nep_kernels();  // kernels_nep.cu: per-device kernel attributes, from cfneb_create
void launch_pending_guard(const Dev &d, int p_first, int count, cudaStream_t st);
void launch_materialize_gen_force(const Dev &d, cudaStream_t st);
void launch_export_dots(const Dev &d, double *dots_out, double *coef_out, cudaStream_t st);
void launch_unpack_neighbors(const Dev &d, int slot, int *count_out, int *list_out, int *shift_out, cudaStream_t st);
void launch_export_path(const Dev &d, double *pos_out, double *cells_out, double *E_out, cudaStream_t st);
void launch_export_state(const Dev &d, double *X_out, double *v_out, cudaStream_t st);
void launch_export_list_state(const Dev &d, double *Xl_out, double *aux_out, cudaStream_t st);  // checkpoint
void launch_import_state(const Dev &d, const double *X_in, const double *v_in, int track, int p_first, int count,
                         cudaStream_t st);  // images p_first .. p_first + count - 1 of the path
void launch_import_aux(const Dev &d, const double *aux_in, int have_aux, int have_fire, double dt, double alpha, int n_pos,
                       int first, unsigned long long steps, cudaStream_t st);
void launch_export_forces(const Dev &d, double *F_out, double *V_out, double *E_out, cudaStream_t st);
double run_fp64_peak(cudaStream_t st);

// ordered-bits helpers for atomicMax on non-negative doubles
__device__ inline unsigned long long nonneg_bits(double x) { return (unsigned long long)__double_as_longlong(x); }
__device__ inline double bits_nonneg(unsigned long long b) { return __longlong_as_double((long long)b); }

// Index t of the first tail bucket whose entries cannot be inside r_cut now: they were built at
// r >= sqrt(r_cut^2 + t (r_list^2 - r_cut^2) / kTailBuckets) and no pair distance has changed by more than acc
// since (Geom::acc, the bound the rebuild decision uses).  kTailBuckets = walk the whole list.
__device__ inline int first_dead_tail_bucket(double r_cut, double r_list, double acc) {
    const double rc2 = r_cut * r_cut, step = (r_list * r_list - rc2) / kTailBuckets;
    const double need = r_cut + acc + 1e-9 * r_cut;
    for (int t = 0; t < kTailBuckets; ++t)
        if (sqrt(rc2 + t * step) >= need) return t;
    return kTailBuckets;
}

// Rows of atom i's (distance-sorted) list that can hold a pair inside r_cut now: everything before the first dead
// tail bucket.  The mirror entry (j; i, -n) of a row below this bound lies below j's bound (same distance, same
// bucket; a pair whose two entries straddle a bucket edge by rounding is out of range by the margin of `need`).
__device__ inline int live_rows(const Dev &d, int slot, int i) {
    const int t_dead = first_dead_tail_bucket(d.r_cut, d.r_list, d.geom[slot].acc);
    return t_dead < kTailBuckets ? (int)d.nbr_tail[((size_t)slot * kTailBuckets + t_dead) * d.Npad + i]
                                 : d.nbr_count[(size_t)slot * d.Npad + i];
}

// Rows of atom i's (distance-sorted) list that can hold a pair inside the angular cut-off now: everything before the
// first kept inner bucket edge that is at least rc_a + acc (built at or beyond that edge, moved by at most acc since:
// the reasoning of live_rows).  All live rows when no kept edge is far enough.
__device__ inline int nep_angular_rows(const Dev &d, int slot, int i) {
    const double rc2 = d.r_cut * d.r_cut, need = d.pot[1] + d.geom[slot].acc + 1e-9 * d.r_cut;
    for (int e = 0; e < kEdgeRows; ++e) {
        const int b = d.edge_b0 + e;
        if (b <= kInnerBuckets && sqrt(rc2 * b / kInnerBuckets) >= need)
            return min((int)d.nbr_edge[((size_t)slot * kEdgeRows + e) * d.Npad + i], d.cap);
    }
    return live_rows(d, slot, i);
}

// 1/sqrt(x) for normal x > 0: hardware seed (2^-22) + one cubically convergent step; no special cases.
__device__ __forceinline__ double rsqrt_nr(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-(x * y), y, 1.0);
    return fma(y * e, fma(0.375, e, 0.5), y);
}

__device__ inline void set_error(Ctl *ctl, int code) { atomicCAS(&ctl->error, 0, code); }

// block-wide sum of NV values per thread; result valid in thread 0. blockDim.x a multiple of 32, <= 1024.
// Fixed tree: the result depends only on the inputs, never on scheduling (bitwise repeatable).
template <int NV>
__device__ inline void block_sum(double (&val)[NV], double *smem /* [32*NV] */) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
#pragma unroll
    for (int q = 0; q < NV; ++q) {
        double x = val[q];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
        if (lane == 0) smem[warp * NV + q] = x;
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int q = 0; q < NV; ++q) {
            double x = (lane < nwarp) ? smem[lane * NV + q] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
            val[q] = x;
        }
    }
    __syncthreads();
}

// Error-free addition (Knuth): s + e = a + b exactly.  Adds only: FMA contraction cannot touch it.
__device__ inline void two_sum(double a, double b, double &s, double &e) {
    s = a + b;
    const double bb = s - a;
    e = (a - (s - bb)) + (b - bb);
}
// (hi, lo) += (h2, l2) in two-double arithmetic (lo stays a small correction; not renormalised)
__device__ inline void dd_add(double &hi, double &lo, double h2, double l2) {
    double s, e;
    two_sum(hi, h2, s, e);
    hi = s;
    lo += l2 + e;
}
// Block-wide sum of one two-double value per thread, same fixed tree as block_sum; result (normalised) in thread 0.
// The image energy is a sum of ~1e5 site energies of the same sign (|E| ~ 9e5 eV at configs[4]) whose DIFFERENCES
// between neighbouring images (~0.3 eV) weight the improved tangent at an extremum (O5): a plain tree loses a few
// ulp(E) ~ 1e-10 in its last levels, which is 1e-9 of those weights.  Carried in two doubles the total is the
// correctly rounded sum of the per-thread values.
__device__ inline void block_sum_dd(double &hi, double &lo, double *smem /* [64] */) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double h2 = __shfl_down_sync(0xffffffffu, hi, o), l2 = __shfl_down_sync(0xffffffffu, lo, o);
        dd_add(hi, lo, h2, l2);
    }
    if (lane == 0) { smem[2 * warp] = hi; smem[2 * warp + 1] = lo; }
    __syncthreads();
    if (warp == 0) {
        hi = (lane < nwarp) ? smem[2 * lane] : 0.0;
        lo = (lane < nwarp) ? smem[2 * lane + 1] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double h2 = __shfl_down_sync(0xffffffffu, hi, o), l2 = __shfl_down_sync(0xffffffffu, lo, o);
            dd_add(hi, lo, h2, l2);
        }
        const double s = hi + lo;  // fast two-sum: |lo| << |hi|
        lo -= s - hi;
        hi = s;
    }
    __syncthreads();
}

__device__ inline double block_max(double x, double *smem /* [32] */) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x = fmax(x, __shfl_down_sync(0xffffffffu, x, o));
    if (lane == 0) smem[warp] = x;
    __syncthreads();
    if (warp == 0) {
        x = (lane < nwarp) ? smem[lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x = fmax(x, __shfl_down_sync(0xffffffffu, x, o));
    }
    __syncthreads();
    return x;  // valid in thread 0
}

}  // namespace cfn

// kernels_neighbor.cu -- K1: per-image cell-list neighbour build under PBC ("neighbors in i's local
// environment under PBC"; O2).  Entry (i; j, n) iff |(s_j - s_i + n) h| < r_list strictly and
// (j, n) != (i, 0), with s = R~ h0^-1 the unwrapped fractional coordinates (Eq. 10), so that the periodic
// shift n is defined relative to the stored coordinates and r^ij = R_j - R_i + n h.
//
// Bins live in wrapped fractional space: axis a has nb_a = floor(w_a / r_list) bins (w_a = perpendicular
// width) and a +-1 stencil when nb_a >= 3, otherwise one bin and explicit shifts m_a in [-reach, reach]
// (boxes smaller than 2 r_list: an atom then sees several periodic images of the same neighbour, itself
// included).  Every kernel exits at once for images whose list is still valid (Geom::rebuild == 0).
//
// Determinism: bins are filled with atomics, then each bin is sorted by atom index, so list order (and with
// it the summation order of the force kernel) is a function of the coordinates only.
//
// Radial order: each atom's list is stored sorted by distance at build time (stable counting sort on 64 buckets
// of r^2).  In a solid the k-th nearest neighbour of every atom of a warp then lies in the same shell, so the
// force kernels' per-entry decisions (inside r_cut? inside the taper zone?) are nearly warp-uniform and are
// taken as warp-level branches with no per-step compaction pass.  The last kTailBuckets buckets divide
// [r_cut^2, r_list^2): the build also stores, per atom, how many entries lie below each of them, and a force
// kernel stops its walk at the first tail bucket that cannot have come inside r_cut yet, given the image's
// accumulated displacement bound Geom::acc (tail_rows()).
#include "cfneb_internal.cuh"

namespace cfn {

__device__ inline bool image_active(const Dev &d, int p_lo, int y, int &slot) {
    int p;
    if (!image_of(y, p_lo, d.ctl->P, p)) return false;
    slot = d.order[p];
    return d.geom[slot].rebuild != 0;
}

// Exclusive scan of the bin populations of one image (one block per image); also primes the fill cursors.
__global__ void __launch_bounds__(1024) bin_scan_kernel(Dev d, int p_lo) {
    int slot;
    if (!image_active(d, p_lo, blockIdx.x, slot)) return;
    const Geom *g = d.geom + slot;
    const int nbins = g->nb[0] * g->nb[1] * g->nb[2];
    int *bc = d.bin_count + (size_t)slot * (d.nbins_max + 1);
    int *cur = d.bin_cursor + (size_t)slot * d.nbins_max;
    const int T = blockDim.x, tid = threadIdx.x;
    const int per = (nbins + T) / T;  // covers nbins + 1 entries
    const int lo = min(tid * per, nbins + 1), hi = min(lo + per, nbins + 1);
    int sum = 0;
    for (int b = lo; b < hi; ++b) sum += bc[b];
    __shared__ int s[1024];
    s[tid] = sum;
    __syncthreads();
    for (int off = 1; off < T; off <<= 1) {
        int t = (tid >= off) ? s[tid - off] : 0;
        __syncthreads();
        s[tid] += t;
        __syncthreads();
    }
    int base = s[tid] - sum;
    for (int b = lo; b < hi; ++b) {
        int c = bc[b];
        bc[b] = base;
        if (b < nbins) cur[b] = base;
        base += c;
    }
}

// (bin_fill and bin_sort run on grids of fixed size over the compact list of rebuilding images, like the search.)
__global__ void __launch_bounds__(kThreadsAtom) bin_fill_kernel(Dev d) {
    const long long total = (long long)d.ctl->n_rebuild * d.N;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int slot = d.rebuild_slots[t / d.N], i = (int)(t % d.N);
        const int bin = d.atom_bin[(size_t)slot * d.Npad + i];
        const int pos = atomicAdd(d.bin_cursor + (size_t)slot * d.nbins_max + bin, 1);
        d.bin_members[(size_t)slot * d.Npad + pos] = i;
    }
}

// One thread per bin: sort the members by atom index, then write the bin-ordered coordinate array.
__global__ void __launch_bounds__(128) bin_sort_kernel(Dev d) {
    const long long total = (long long)d.ctl->n_rebuild * d.nbins_max;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
    const int slot = d.rebuild_slots[t / d.nbins_max], b = (int)(t % d.nbins_max);
    const Geom *g = d.geom + slot;
    const int nbins = g->nb[0] * g->nb[1] * g->nb[2];
    if (b >= nbins) continue;
    const int *bc = d.bin_count + (size_t)slot * (d.nbins_max + 1);
    int *mem = d.bin_members + (size_t)slot * d.Npad;
    const int lo = bc[b], hi = bc[b + 1];
    for (int q = lo + 1; q < hi; ++q) {  // insertion sort (bins hold a few tens of atoms)
        int x = mem[q], r = q - 1;
        while (r >= lo && mem[r] > x) { mem[r + 1] = mem[r]; --r; }
        mem[r + 1] = x;
    }
    const double4 *Sw = d.Sw + (size_t)slot * d.Npad;
    double4 *out = d.binned + (size_t)slot * d.Npad;
    float4 *outc = d.binned_c + (size_t)slot * d.Npad;
    for (int q = lo; q < hi; ++q) {
        const int i = mem[q];
        double4 w = Sw[i];
        unsigned long long fl = (unsigned long long)__double_as_longlong(w.w);
        w.w = __longlong_as_double((long long)((unsigned long long)i | (fl << kShiftBits)));
        out[q] = w;
        // fp32 Cartesian copy of the wrapped position for the search's prefilter
        outc[q] = make_float4((float)(w.x * g->h[0] + w.y * g->h[3] + w.z * g->h[6]),
                              (float)(w.x * g->h[1] + w.y * g->h[4] + w.z * g->h[7]),
                              (float)(w.x * g->h[2] + w.y * g->h[5] + w.z * g->h[8]), 0.f);
    }
    }  // work items
}

__device__ inline void stencil_axis(int nb, int bi, int dlt, int &bj, int &m) {
    if (nb >= 3) {
        int t = bi + dlt;
        m = (t < 0) ? -1 : (t >= nb ? 1 : 0);
        bj = t - m * nb;
    } else {
        bj = 0;
        m = dlt;
    }
}

// Compact list of the images (slots) of the selected set whose list is rebuilt this step, in path order.
__global__ void __launch_bounds__(256) rebuild_list_kernel(Dev d, int p_lo) {
    const int P = d.ctl->P;
    const int ny = images_in_grid(d.S, p_lo);
    __shared__ int s_warp[8], s_base;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_base = 0;
    __syncthreads();
    for (int y0 = 0; y0 < ny; y0 += 256) {  // 256 images per round, compacted in path order
        const int y = y0 + threadIdx.x;
        int p, slot = -1;
        bool on = false;
        if (y < ny && image_of(y, p_lo, P, p)) {
            slot = d.order[p];
            on = d.geom[slot].rebuild != 0;
        }
        const unsigned m = __ballot_sync(0xffffffffu, on);
        if (lane == 0) s_warp[warp] = __popc(m);
        __syncthreads();
        int off = s_base;
        for (int w = 0; w < warp; ++w) off += s_warp[w];
        if (on) d.rebuild_slots[off + __popc(m & ((1u << lane) - 1u))] = slot;
        __syncthreads();
        if (threadIdx.x == 0) {
            int t = 0;
            for (int w = 0; w < 8; ++w) t += s_warp[w];
            s_base += t;
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) d.ctl->n_rebuild = s_base;
}

constexpr int kRadialBuckets = kInnerBuckets + kTailBuckets;
#ifndef CFNEB_K1_DRAIN
#define CFNEB_K1_DRAIN 4
#endif
#ifndef CFNEB_K1_SCAN
#define CFNEB_K1_SCAN 8
#endif
constexpr int kDrain = CFNEB_K1_DRAIN, kScan = CFNEB_K1_SCAN;  // candidates per round of the drain / of the prefilter scan
constexpr uint32_t kCodeFar = 0u | (4u << 3) | (4u << 6);
#ifndef CFNEB_SEARCH_BLOCKS
#define CFNEB_SEARCH_BLOCKS 6
#endif
// Round 2: the grid has a fixed size (CFNEB_SEARCH_BLOCKS blocks per multiprocessor) and takes its work items
// (rebuilding image, block of 128 atoms) from the compact list of rebuild_list_kernel -- a step in which no list is
// stale costs one exit per resident block instead of 77 616 -- and the scratch of a block (the candidate queue, which
// the drain rewrites in place as the unsorted column, and the buckets: scr_queue, scr_bkt, 160 KB per block at cap 224)
// is a region of its own, reused item after item, instead of arrays of the size of the list itself (round 1: 11.4 GB of workspace).  The candidates that pass the
// fp32 prefilter are queued for the whole environment and drained once (see `queue` below): 0.56 -> 0.43 ms per image
// at c4; with the queue out of shared memory six blocks are resident (0.40) and the scan reads past short bins
// instead of clamping its index (0.38); unsorted column written over the queue (0.355).
//
// One thread per atom, two phases per warp so that lanes stay converged:
//   scan   every lane walks the same stencil cell (its own bin range of it) kScan candidates at a time -- independent
//          fp32 loads, a prefilter on fp32 Cartesian coordinates against r_list + margin -- and appends the survivors
//          (about one in six) to its column of the block's candidate queue in global scratch ([row][thread]);
//   drain  once per atom, after the whole stencil (earlier only if a lane's column is about to run out of rows, which
//          takes more candidates than the list has capacity): all lanes in step, kDrain candidates per round, the exact
//          fp64 test |ds h|^2 < r_list^2, which alone decides membership, and the accepted (j | code << 23) with its
//          r^2 bucket written over the queue rows already read (the unsorted column) and to scr_bkt; histogram of the
//          buckets in shared memory.
// The column is then counting-sorted into nbr_list.  Rows cnt..cap-1 are filled with a stand-in entry (the atom itself
// shifted by -4 cell vectors along axis 0: farther than r_list whenever a list can be built at all), so the force
// kernels read any row below cap without a bounds test and find it out of range.
__global__ void __launch_bounds__(kThreadsAtom, CFNEB_SEARCH_BLOCKS) neighbor_search_kernel(Dev d) {
    __shared__ unsigned short s_hist[kRadialBuckets * kThreadsAtom];
    __shared__ int s_max;
    if (threadIdx.x == 0) s_max = 0;
    __syncthreads();  // before any thread's atomicMax on it
    const int n_items = d.ctl->n_rebuild * d.nblk_atom;
    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
    const int slot = d.rebuild_slots[item / d.nblk_atom];
    const int i = (item % d.nblk_atom) * blockDim.x + threadIdx.x;
    const bool valid = i < d.N;
    const int ic = valid ? i : 0;  // idle lanes shadow atom 0 with empty bin ranges
    int cnt = 0;
    bool bad_shift = false;
    unsigned short *hist = s_hist + threadIdx.x;
    // candidates that pass the prefilter wait in a queue long enough for a whole environment (global scratch of the
    // block, L2-resident): ONE drain per atom.  With a 32-entry queue in shared memory the drain ran whenever any
    // lane's queue was full, the average lane a third full: 413 rounds per warp for 153 neighbours per atom at c4.
    const int kQueue = d.cap + kQueueSlack;
    uint32_t *queue = d.scr_queue + (size_t)blockIdx.x * kQueue * kThreadsAtom + threadIdx.x;
    for (int b = 0; b < kRadialBuckets; ++b) hist[b * kThreadsAtom] = 0;
    const Geom *g = d.geom + slot;
    const int nb0 = g->nb[0], nb1 = g->nb[1], nb2 = g->nb[2];
    const int re0 = g->reach[0], re1 = g->reach[1], re2 = g->reach[2];
    if (re0 > 3 || re1 > 3 || re2 > 3) {  // periodic shifts are stored in 3 bits per axis
        if (threadIdx.x == 0) set_error(d.ctl, CFNEB_ECELL);
        continue;
    }
    double h[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) h[k] = g->h[k];
    const double4 si = d.Sw[(size_t)slot * d.Npad + ic];
    const unsigned long long fli = (unsigned long long)__double_as_longlong(si.w);
    const int fi0 = (int)(fli & 1023u), fi1 = (int)((fli >> 10) & 1023u), fi2 = (int)((fli >> 20) & 1023u);
    const int bin = d.atom_bin[(size_t)slot * d.Npad + ic];
    const int bi0 = bin / (nb1 * nb2), bi1 = (bin / nb2) % nb1, bi2 = bin % nb2;
    const int *__restrict__ bc = d.bin_count + (size_t)slot * (d.nbins_max + 1);
    const double4 *__restrict__ binned = d.binned + (size_t)slot * d.Npad;
    const float4 *__restrict__ binned_c = d.binned_c + (size_t)slot * d.Npad;
    // prefilter margin: rounding of fp32 coordinates of magnitude <= L = the cell's extent including the shifts
    // (fp32 eps 1.2e-7; 64 eps L is > 10x the worst case of the 3 subtractions and 3 products)
    const float cix = (float)(si.x * h[0] + si.y * h[3] + si.z * h[6]), ciy = (float)(si.x * h[1] + si.y * h[4] + si.z * h[7]),
                ciz = (float)(si.x * h[2] + si.y * h[5] + si.z * h[8]);
    double Lext = 0.0;
    for (int k = 0; k < 9; ++k) Lext += fabs(h[k]);
    const float rlf = (float)(d.r_list + 64.0 * 1.2e-7 * 2.0 * Lext * (1.0 + max(re0, max(re1, re2))));
    const float rl2f = rlf * rlf;
    uint32_t *__restrict__ list = d.nbr_list + (size_t)slot * d.cap * d.Npad + ic;
    // The drain writes its accepted entries over the queue rows it has already read: the unsorted column is rows
    // 0..cnt-1 of the queue.  Waiting candidates occupy rows q0..nq-1; q0 = 0 until a drain has run, then the number of
    // accepted entries, so that candidates queued after a mid-scan drain land behind the column, not on it, and the
    // drain's write row (cnt) never passes its read row (q0 + c: at most c entries were accepted since q0 = cnt).
    uint32_t *tmp = queue;
    unsigned char *__restrict__ bkt = d.scr_bkt + (size_t)blockIdx.x * d.cap * kThreadsAtom + threadIdx.x;
    // radial buckets: kInnerBuckets uniform in r^2 below r_cut^2, kTailBuckets uniform between r_cut^2 and r_list^2
    const double rl2 = d.r_list * d.r_list, rc2 = d.r_cut * d.r_cut;
    const double bscale_in = (double)kInnerBuckets / rc2, bscale_tail = rl2 > rc2 ? (double)kTailBuckets / (rl2 - rc2) : 0.0;
    int nq = 0, q0 = 0;

    auto flush = [&]() {
        const int nw = nq - q0;  // this lane's waiting candidates
        const int nq_w = __reduce_max_sync(0xffffffffu, nw);
        // kDrain candidates per round: their queue entries and coordinates are requested together (the walk is
        // bound by the latency of these two dependent loads, not by their number)
        for (int c0 = 0; c0 < nq_w; c0 += kDrain) {
          uint32_t ee[kDrain];
          double4 cc[kDrain];
#pragma unroll
          for (int u = 0; u < kDrain; ++u) ee[u] = queue[min(q0 + c0 + u, kQueue - 1) * kThreadsAtom];
#pragma unroll
          for (int u = 0; u < kDrain; ++u) cc[u] = binned[c0 + u < nw ? (int)(ee[u] & kIdxMask) : ic];
#pragma unroll
          for (int u = 0; u < kDrain; ++u) {
            const int c = c0 + u;
            if (c >= nw) continue;
            const uint32_t e = ee[u];
            const int m0 = (int)((e >> kShiftBits) & 7u) - 4, m1 = (int)((e >> (kShiftBits + 3)) & 7u) - 4,
                      m2 = (int)((e >> (kShiftBits + 6)) & 7u) - 4;
            const double4 c4 = cc[u];
            const double s0 = c4.x - si.x + (double)m0, s1 = c4.y - si.y + (double)m1, s2 = c4.z - si.z + (double)m2;
            const double rx = s0 * h[0] + s1 * h[3] + s2 * h[6];
            const double ry = s0 * h[1] + s1 * h[4] + s2 * h[7];
            const double rz = s0 * h[2] + s1 * h[5] + s2 * h[8];
            const double r2 = rx * rx + ry * ry + rz * rz;
            if (!(r2 < rl2)) continue;
            const unsigned long long pk = (unsigned long long)__double_as_longlong(c4.w);
            const int j = (int)(pk & kIdxMask);
            const int n0 = m0 - (int)((pk >> kShiftBits) & 1023u) + fi0;
            const int n1 = m1 - (int)((pk >> (kShiftBits + 10)) & 1023u) + fi1;
            const int n2 = m2 - (int)((pk >> (kShiftBits + 20)) & 1023u) + fi2;
            if (j == i && n0 == 0 && n1 == 0 && n2 == 0) continue;
            if (cnt < d.cap) {
                if (n0 < -4 || n0 > 3 || n1 < -4 || n1 > 3 || n2 < -4 || n2 > 3) bad_shift = true;
                if (n0 == -4 && n1 == 0 && n2 == 0) bad_shift = true;  // reserved for the stand-in entry
                const uint32_t code = (uint32_t)((n0 + 4) & 7) | ((uint32_t)((n1 + 4) & 7) << 3) |
                                      ((uint32_t)((n2 + 4) & 7) << 6);
                const int bk = r2 < rc2 ? min((int)(r2 * bscale_in), kInnerBuckets - 1)
                                        : kInnerBuckets + min((int)((r2 - rc2) * bscale_tail), kTailBuckets - 1);
                tmp[(size_t)cnt * kThreadsAtom] = (uint32_t)j | (code << kShiftBits);
                bkt[(size_t)cnt * kThreadsAtom] = (unsigned char)bk;
                hist[bk * kThreadsAtom] += 1;
            }
            ++cnt;
          }
        }
        nq = q0 = min(cnt, d.cap);
    };

    for (int d0 = -re0; d0 <= re0; ++d0) {
        int bj0, m0;
        stencil_axis(nb0, bi0, d0, bj0, m0);
        for (int d1 = -re1; d1 <= re1; ++d1) {
            int bj1, m1;
            stencil_axis(nb1, bi1, d1, bj1, m1);
            for (int d2 = -re2; d2 <= re2; ++d2) {
                int bj2, m2;
                stencil_axis(nb2, bi2, d2, bj2, m2);
                const int b = (bj0 * nb1 + bj1) * nb2 + bj2;
                const int lo = bc[b], hi = valid ? bc[b + 1] : lo;
                const int len_w = __reduce_max_sync(0xffffffffu, hi - lo);
                const uint32_t mcode = ((uint32_t)(m0 + 4) | ((uint32_t)(m1 + 4) << 3) | ((uint32_t)(m2 + 4) << 6)) << kShiftBits;
                // own position minus the periodic shift of this stencil cell, fp32
                const float ox = cix - (float)(m0 * h[0] + m1 * h[3] + m2 * h[6]), oy = ciy - (float)(m0 * h[1] + m1 * h[4] + m2 * h[7]),
                            oz = ciz - (float)(m0 * h[2] + m1 * h[5] + m2 * h[8]);
                for (int t = 0; t < len_w; t += kScan) {
                    float4 cf[kScan];
#pragma unroll
                    // (reads past this lane's bin are masked by q < hi below; they stay inside the array and its slack)
                    for (int u = 0; u < kScan; ++u) cf[u] = binned_c[lo + t + u];
#pragma unroll
                    for (int u = 0; u < kScan; ++u) {
                        const int q = lo + t + u;
                        const float fx = cf[u].x - ox, fy = cf[u].y - oy, fz = cf[u].z - oz;
                        if (q < hi && fx * fx + fy * fy + fz * fz < rl2f) {
                            queue[nq * kThreadsAtom] = (uint32_t)q | mcode;
                            ++nq;
                        }
                    }
                    if (__any_sync(0xffffffffu, nq > kQueue - kScan)) flush();
                }
            }
        }
    }
    flush();
    if (valid) {
    const int n = min(cnt, d.cap);
    d.nbr_count[(size_t)slot * d.Npad + i] = n;
    // stable counting sort by r^2 bucket: exclusive starts, then placement (scan order kept inside a bucket),
    // four entries per round so that the global loads of a round are independent
    int start = 0;
    unsigned short *tail = d.nbr_tail + (size_t)slot * kTailBuckets * d.Npad + i;
    unsigned short *edge = d.nbr_edge ? d.nbr_edge + (size_t)slot * kEdgeRows * d.Npad + i : nullptr;
    for (int b = 0; b < kRadialBuckets; ++b) {
        const int c = hist[b * kThreadsAtom];
        hist[b * kThreadsAtom] = (unsigned short)start;
        if (edge && (unsigned)(b - d.edge_b0) < (unsigned)kEdgeRows) edge[(size_t)(b - d.edge_b0) * d.Npad] = (unsigned short)start;
        if (b >= kInnerBuckets) tail[(size_t)(b - kInnerBuckets) * d.Npad] = (unsigned short)start;  // entries below tail bucket b - 56
        start += c;
    }
    for (int k0 = 0; k0 < n; k0 += 4) {
        uint32_t t[4];
        int bk[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const size_t o = (size_t)min(k0 + u, n - 1) * kThreadsAtom;
            t[u] = tmp[o];
            bk[u] = bkt[o];
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (k0 + u >= n) break;
            unsigned short &cur = hist[bk[u] * kThreadsAtom];
            list[(size_t)cur * d.Npad] = t[u];
            cur += 1;
        }
    }
    }  // valid
    {   // stand-in rows cnt..cap-1 (idle lanes of the last block included: their columns exist up to Npad)
        const int i_pad = i;
        if (i_pad < d.Npad) {
            uint32_t *col = d.nbr_list + (size_t)slot * d.cap * d.Npad + i_pad;
            const uint32_t far = (uint32_t)(valid ? i : 0) | (kCodeFar << kShiftBits);
            for (int k = valid ? min(cnt, d.cap) : 0; k < d.cap; ++k) col[(size_t)k * d.Npad] = far;
        }
    }
    if (cnt > d.cap_user) set_error(d.ctl, CFNEB_ENEIGH_OVERFLOW);
    if (bad_shift) set_error(d.ctl, CFNEB_ECELL);
    atomicMax(&s_max, cnt);
    }  // work items
    // block-level max, then one atomic per block
    __syncthreads();
    if (threadIdx.x == 0 && s_max > d.ctl->max_nbr_seen) atomicMax(&d.ctl->max_nbr_seen, s_max);
}

// Parity hook: list of one slot in the external layout count[N], list[N][cap] (-1 padded), shift[N][cap][3].
__global__ void unpack_neighbors_kernel(Dev d, int slot, int *count_out, int *list_out, int *shift_out) {
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (size_t)d.N * d.cap_user) return;
    const int i = (int)(t / d.cap_user), k = (int)(t % d.cap_user);  // internal (storage-order) atom index
    const size_t e = (size_t)d.perm[i] * d.cap_user + k;             // row of the caller's atom
    const int c = d.nbr_count[(size_t)slot * d.Npad + i];
    if (k == 0) count_out[d.perm[i]] = c;
    int j = -1, n0 = 0, n1 = 0, n2 = 0;
    if (k < c) {
        const uint32_t w = d.nbr_list[((size_t)slot * d.cap + k) * d.Npad + i];
        j = d.perm[w & kIdxMask];
        const uint32_t code = w >> kShiftBits;
        n0 = (int)(code & 7u) - 4;
        n1 = (int)((code >> 3) & 7u) - 4;
        n2 = (int)((code >> 6) & 7u) - 4;
    }
    list_out[e] = j;
    shift_out[3 * e] = n0;
    shift_out[3 * e + 1] = n1;
    shift_out[3 * e + 2] = n2;
}

void launch_neighbor_build(const Dev &d, int p_lo, cudaStream_t st) {
    const int nimg = images_in_grid(d.S, p_lo);
    if (nimg <= 0) return;
    rebuild_list_kernel<<<1, 256, 0, st>>>(d, p_lo);
    bin_scan_kernel<<<nimg, 1024, 0, st>>>(d, p_lo);
    bin_fill_kernel<<<d.n_sm * 8, kThreadsAtom, 0, st>>>(d);
    bin_sort_kernel<<<d.n_sm * 8, 128, 0, st>>>(d);
    neighbor_search_kernel<<<d.n_search_blocks, kThreadsAtom, 0, st>>>(d);
    if (d.potential == CFNEB_POT_SW || d.potential == CFNEB_POT_DNN || d.potential == CFNEB_POT_NEP) launch_mirror_sw(d, p_lo, st);
}

int search_blocks_per_sm() { return CFNEB_SEARCH_BLOCKS; }

void launch_unpack_neighbors(const Dev &d, int slot, int *count_out, int *list_out, int *shift_out, cudaStream_t st) {
    const size_t n = (size_t)d.N * d.cap_user;
    unpack_neighbors_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d, slot, count_out, list_out, shift_out);
}

}  // namespace cfn

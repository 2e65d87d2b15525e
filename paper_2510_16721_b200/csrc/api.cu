// api.cu -- the C ABI of include/cfneb.h: handle, workspace carving, CUDA-graph capture of one CFNEB
// iteration (K0-K6), host-side image control (O9) and the parity / checkpoint hooks.
// All arithmetic of the method runs in the kernels; this file only marshals, launches and copies.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "cfneb_internal.cuh"

using namespace cfn;

static thread_local char g_cuda_err[512] = "";

#define CK(call)                                                                                       \
    do {                                                                                               \
        cudaError_t e_ = (call);                                                                       \
        if (e_ != cudaSuccess) {                                                                       \
            snprintf(g_cuda_err, sizeof g_cuda_err, "%s at %s:%d: %s", #call, __FILE__, __LINE__,     \
                     cudaGetErrorString(e_));                                                          \
            return CFNEB_ECUDA;                                                                        \
        }                                                                                              \
    } while (0)

struct cfneb {
    Dev d;
    cfneb_params prm;
    cudaStream_t st;
    bool own_stream;
    int P;
    std::vector<int> order;  // host mirror of the order table (only the host edits it)
    std::vector<int> free_slots;
    cudaGraph_t graph;
    cudaGraphExec_t exec;
    int graph_nodes;
    bool mirror_dirty;    // the device edited P / order / free slots (cfneb_step_adaptive); host mirrors are stale
    bool interior_stale;  // cfneb_set_path replaced the path and the interior images have not been evaluated since
    int device;           // CUDA device the workspace and the stream live on (current at cfneb_create)
    cudaStream_t st2;     // copy stream of cfneb_step_hosted (created on first use)
    std::vector<cudaEvent_t> ev_blocks;  // one event per image block of cfneb_step_hosted
};

// Every ABI entry runs with the handle's device current and puts the caller's back on return, so a handle on
// cuda:1 works while cuda:0 is current.
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(const cfneb *h) {
        int cur = -1;
        if (h && cudaGetDevice(&cur) == cudaSuccess && cur != h->device && cudaSetDevice(h->device) == cudaSuccess) prev = cur;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
    DeviceGuard(const DeviceGuard &) = delete;
    DeviceGuard &operator=(const DeviceGuard &) = delete;
};

// ---- workspace carving (one function serves the size query and create) ----
namespace {
struct Carver {
    char *base;
    size_t off;
    template <typename T>
    T *take(size_t n) {
        off = (off + 255) & ~(size_t)255;
        T *p = base ? reinterpret_cast<T *>(base + off) : nullptr;
        off += n * sizeof(T);
        return p;
    }
};

double cutoff_of(const cfneb_params *prm) {
    switch (prm->potential) {
        case CFNEB_POT_LJ_SF: return prm->pot[2];
        case CFNEB_POT_SW: return prm->pot[2] * prm->pot[1];
        case CFNEB_POT_DNN: return prm->pot[0];
        case CFNEB_POT_NEP: return prm->pot[0];  // the radial (larger) cut-off
        default: return prm->pot[7];
    }
}

bool many_body(const cfneb_params *prm) {
    return prm->potential == CFNEB_POT_SW || prm->potential == CFNEB_POT_DNN || prm->potential == CFNEB_POT_NEP;
}

bool valid_params(int32_t n_atoms, const cfneb_params *prm) {
    if (!prm || n_atoms < 1 || n_atoms >= kMaxAtoms) return false;
    if (prm->potential < CFNEB_POT_LJ_SF || prm->potential > CFNEB_POT_NEP) return false;
    if (prm->cell_mode < CFNEB_CELL_FIXED || prm->cell_mode > CFNEB_CELL_D) return false;
    if (prm->max_images < 3 || prm->max_neighbors < 1 || prm->max_neighbors > 4096) return false;
    if (!(prm->skin >= 0.0) || !(prm->cell_factor >= 0.0) || !isfinite(prm->pressure)) return false;
    const double rc = cutoff_of(prm);
    if (!(rc > 0.0)) return false;
    if (prm->potential == CFNEB_POT_DNN) {
        const double *q = prm->pot;
        for (int k = 1; k <= 5; ++k)
            if (!(q[k] >= 0.0) || q[k] != floor(q[k]) || q[k] > 9.0e15) return false;
        if (q[1] < 1 || q[1] > 4 || q[2] < 1 || q[2] > 4 || q[3] < 1 || q[3] > 3 || q[4] < 1 || q[4] > 8) return false;
    }
    if (prm->potential == CFNEB_POT_NEP) {
        const double *q = prm->pot;
        for (int k = 2; k <= 9; ++k)
            if (!(q[k] >= 0.0) || q[k] != floor(q[k]) || q[k] > 9.0e15) return false;
        if (!(q[1] > 0.0) || q[1] > q[0]) return false;                                        // rc_a <= rc_r
        if (q[2] < 1 || q[2] > 8 || q[3] < 1 || q[3] > 8 || q[4] < 1 || q[4] > 12 || q[5] < 1 || q[5] > 12) return false;
        if (q[6] < 1 || q[6] > 4 || q[7] < 1 || q[7] > 64 || q[8] < 1 || q[8] > 2) return false;
    }
    if (prm->potential == CFNEB_POT_FS_MORSE && !(prm->pot[7] > prm->pot[6])) return false;
    if (!(prm->fire_dt0 > 0.0) || !(prm->fire_dtmax > 0.0) || !(prm->fire_maxstep > 0.0)) return false;
    return true;
}

size_t carve(int32_t N, const cfneb_params *prm, void *base, Dev *out) {
    Dev d;
    memset(&d, 0, sizeof d);
    d.N = N;
    d.Npad = (N + 31) / 32 * 32;
    d.S = prm->max_images;
    d.cap = (prm->max_neighbors + 1) & ~1;  // even: the pair kernels walk two rows per iteration without a bound check
    d.cap_user = prm->max_neighbors;
    d.nblk_atom = (N + kThreadsAtom - 1) / kThreadsAtom;
    d.nblk_force = prm->potential == CFNEB_POT_NEP ? (N + 31) / 32 : many_body(prm) ? d.nblk_atom : (N + kThreadsPair - 1) / kThreadsPair;
    d.nblk_stream = (d.Npad + kAtomsPerStreamBlock - 1) / kAtomsPerStreamBlock;
    d.nbins_max = N > 64 ? N : 64;
    const size_t S = d.S, Npad = d.Npad, img = 3 * Npad;
    Carver c{static_cast<char *>(base), 0};
    d.ctl = c.take<Ctl>(1);
    d.order = c.take<int>(S);
    d.free_stack = c.take<int>(S);
    d.seglen = c.take<double>(2 * S);
    d.hist = c.take<double>((size_t)kHistLen * kHistFields);
    d.plan_q = c.take<int>(S);
    d.plan_t = c.take<double>(S);
    d.perm = c.take<int>(Npad);
    d.geom = c.take<Geom>(S);
    d.X = c.take<double>(2 * S * img);
    d.v = c.take<double>(S * img);
    d.F = c.take<double>(S * img);
    d.Rc = c.take<double4>(S * Npad);
    d.Sw = c.take<double4>(S * Npad);
    d.binned = c.take<double4>(S * Npad);
    // + slack: the prefilter scan reads (masked) past a short bin's end, by at most the longest bin of the warp's
    // stencil; a bin of the coarsest grid (3 r_list wide on two axes) holds fewer than 4 x cap atoms
    d.binned_c = c.take<float4>(S * Npad + 4096 + 8 * (size_t)d.cap);
    d.Xc = c.take<double>(2 * S * 9);
    d.vc = c.take<double>(S * 9);
    d.E = c.take<double>(S);
    d.V = c.take<double>(S * 9);
    d.Gc = c.take<double>(S * 9);
    d.dots = c.take<double>(S * kNDots);
    d.coef = c.take<double>(S * 4);
    d.part_force = c.take<double>(S * d.nblk_force * kNForcePart);
    d.part_dots = c.take<double>(S * d.nblk_stream * kNDots);
    d.relax = c.take<RelaxState>(2);
    d.part_relax = c.take<double>((size_t)2 * d.nblk_stream * 4);
    d.dispmax = c.take<unsigned long long>(S);
    d.dispmax_in = c.take<unsigned long long>(S);
    d.disptot = c.take<unsigned long long>(S);
    d.Xb = c.take<double>(S * img);
    d.Xcb = c.take<double>(S * 9);
    d.nbr_count = c.take<int>(S * Npad);
    d.nbr_list = c.take<uint32_t>(S * (size_t)d.cap * Npad + 16 * Npad);  // 16 rows of slack for the force kernels' look-ahead
    d.nbr_tail = c.take<unsigned short>(S * (size_t)kTailBuckets * Npad);
    d.nbr_edge = prm->potential == CFNEB_POT_NEP ? c.take<unsigned short>(S * (size_t)kEdgeRows * Npad) : nullptr;
    d.rebuild_slots = c.take<int>(S);
    {   // K1 scratch: one region per resident block of the search kernel.  The SIZE is that of a fixed upper bound on
        // the multiprocessor count (sm_100a parts have 148 or fewer), so that cfneb_workspace_bytes does not depend on
        // which device -- if any -- is current when it is asked; the GRID uses the device that is current at
        // cfneb_create, clamped to what the scratch holds.
        constexpr int kScratchSMs = 160;
        int dev = 0, sms = 148;
        if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        else cudaGetLastError();
        d.n_sm = sms;
        d.n_search_blocks = (sms < kScratchSMs ? sms : kScratchSMs) * search_blocks_per_sm();
        const size_t nscr = (size_t)kScratchSMs * search_blocks_per_sm();
        d.scr_bkt = c.take<unsigned char>(nscr * d.cap * kThreadsAtom);
        d.scr_queue = c.take<uint32_t>(nscr * (d.cap + kQueueSlack) * kThreadsAtom);
    }
    d.part = many_body(prm) ? c.take<double>(S * (size_t)d.cap * 3 * Npad) : nullptr;
    d.nbr_mirror = many_body(prm) ? c.take<unsigned short>(S * (size_t)d.cap * Npad) : nullptr;
    d.dn_w = prm->potential == CFNEB_POT_DNN ? c.take<double>(kDnWeights)
             : prm->potential == CFNEB_POT_NEP ? c.take<double>(nep_weight_count(prm->pot)) : nullptr;
    d.types = prm->potential == CFNEB_POT_NEP ? c.take<int>(Npad) : nullptr;
    d.nep_q = prm->potential == CFNEB_POT_NEP ? c.take<double>(S * (size_t)8 * Npad) : nullptr;
    d.nep_kr_pad = prm->potential == CFNEB_POT_NEP ? nep_kr_padded(prm->pot) : 0;
    d.nep_w = prm->potential == CFNEB_POT_NEP ? c.take<double>(S * (size_t)Npad * (size_t)prm->pot[8] * d.nep_kr_pad) : nullptr;
    d.nep_S = prm->potential == CFNEB_POT_NEP ? c.take<double>(S * (size_t)prm->pot[3] * 35 * Npad) : nullptr;
    d.bin_count = c.take<int>(S * ((size_t)d.nbins_max + 1));
    d.bin_cursor = c.take<int>(S * (size_t)d.nbins_max);
    d.bin_members = c.take<int>(S * Npad);
    d.atom_bin = c.take<int>(S * Npad);
    // scratch = two halves; a half holds one exported array set (P x (N+3) x 3, or P x N x 3 + P x 9 + P)
    const size_t half = S * ((size_t)(N + 3) * 3 + 16) * sizeof(double);
    size_t sb = 2 * half + 1024;
    const size_t nb = (size_t)N * d.cap_user * 4 * sizeof(int) + (size_t)N * sizeof(int) + 1024;
    if (nb > sb) sb = nb;
    d.scratch = c.take<char>(sb);
    d.scratch_bytes = sb;
    d.fneb = base ? reinterpret_cast<double *>(static_cast<char *>(d.scratch) + half) : nullptr;
    if (out) *out = d;
    return (c.off + 255) & ~(size_t)255;
}

void perp_widths(const double *h, double *w) {
    const double vol = fabs(det3(h));
    for (int a = 0; a < 3; ++a) {
        const double *b = h + 3 * ((a + 1) % 3), *c = h + 3 * ((a + 2) % 3);
        const double cx = b[1] * c[2] - b[2] * c[1], cy = b[2] * c[0] - b[0] * c[2], cz = b[0] * c[1] - b[1] * c[0];
        w[a] = vol / sqrt(cx * cx + cy * cy + cz * cz);
    }
}

// Spatial storage order: Morton order of a grid of edge ~ r_list / 2 over the initial endpoint (ties by the
// caller's index).  perm[internal] = caller's index.  Any order is correct; this one keeps the neighbours of
// consecutive atoms close in memory.
void spatial_order(int N, const double *pos, const double *cell, double r_list, std::vector<int> &perm) {
    double inv[9], w[3];
    inv3(cell, inv);
    perp_widths(cell, w);
    int n[3];
    for (int a = 0; a < 3; ++a) n[a] = std::max(1, std::min(1023, (int)floor(w[a] / (0.5 * r_list))));
    std::vector<unsigned long long> key(N);
    for (int i = 0; i < N; ++i) {
        const double *r = pos + 3 * (size_t)i;
        unsigned c[3];
        for (int a = 0; a < 3; ++a) {
            double s = r[0] * inv[a] + r[1] * inv[3 + a] + r[2] * inv[6 + a];
            s -= floor(s);
            int b = (int)(s * n[a]);
            c[a] = (unsigned)std::max(0, std::min(n[a] - 1, std::isfinite(s) ? b : 0));
        }
        unsigned long long m = 0;
        for (int bit = 0; bit < 10; ++bit)
            for (int a = 0; a < 3; ++a) m |= (unsigned long long)((c[a] >> bit) & 1u) << (3 * bit + a);
        key[i] = m;
    }
    perm.resize(N);
    for (int i = 0; i < N; ++i) perm[i] = i;
    std::stable_sort(perm.begin(), perm.end(), [&](int a, int b) { return key[a] < key[b]; });
}

int device_error(cfneb *h, int *code) {
    CK(cudaMemcpyAsync(code, &h->d.ctl->error, sizeof(int), cudaMemcpyDeviceToHost, h->st));
    CK(cudaStreamSynchronize(h->st));
    return CFNEB_OK;
}

int sync_status(cfneb *h) {  // synchronise; surface launch errors and the sticky device error
    int code = 0;
    int rc = device_error(h, &code);
    if (rc) return rc;
    CK(cudaGetLastError());
    return code;
}

void enqueue_step(cfneb *h, cudaEvent_t *ev) {
    const Dev &d = h->d;
    cudaStream_t st = h->st;
    if (ev) cudaEventRecord(ev[0], st);
    launch_cell_prep(d, 1, MODE_STEP, st);
    if (ev) cudaEventRecord(ev[1], st);
    launch_neighbor_build(d, 1, st);
    if (ev) cudaEventRecord(ev[2], st);
    launch_force(d, 1, st);
    launch_finalize(d, 1, st);  // E, V, G_cell from the force partials: part of the force evaluation
    if (ev) cudaEventRecord(ev[3], st);
    launch_reduce(d, st);
    if (ev) cudaEventRecord(ev[4], st);
    launch_scalar(d, 0, st);
    if (ev) cudaEventRecord(ev[5], st);
    launch_update(d, st);
    if (ev) cudaEventRecord(ev[6], st);
}

// Evaluate every image once at the current X (endpoint energies; fresh neighbour lists).
void enqueue_evaluate_all(cfneb *h) {
    const Dev &d = h->d;
    launch_cell_prep(d, 0, MODE_STEP, h->st);
    launch_neighbor_build(d, 0, h->st);
    launch_force(d, 0, h->st);
    launch_finalize(d, 0, h->st);
}

int force_rebuild_all(cfneb *h) {
    std::vector<Geom> g(h->d.S);
    CK(cudaMemcpyAsync(g.data(), h->d.geom, sizeof(Geom) * h->d.S, cudaMemcpyDeviceToHost, h->st));
    CK(cudaStreamSynchronize(h->st));
    for (auto &x : g) { x.force_rebuild = 1; x.acc = 0.0; x.since = 0; }
    CK(cudaMemcpyAsync(h->d.geom, g.data(), sizeof(Geom) * h->d.S, cudaMemcpyHostToDevice, h->st));
    CK(cudaStreamSynchronize(h->st));
    return CFNEB_OK;
}

int upload_order(cfneb *h) {
    std::vector<int> full(h->d.S, 0), fs(h->d.S, 0);
    for (int p = 0; p < h->P; ++p) full[p] = h->order[p];
    const int n_free = (int)h->free_slots.size();
    for (int k = 0; k < n_free; ++k) fs[k] = h->free_slots[k];
    CK(cudaMemcpyAsync(h->d.order, full.data(), sizeof(int) * h->d.S, cudaMemcpyHostToDevice, h->st));
    CK(cudaMemcpyAsync(h->d.free_stack, fs.data(), sizeof(int) * h->d.S, cudaMemcpyHostToDevice, h->st));
    CK(cudaMemcpyAsync(&h->d.ctl->P, &h->P, sizeof(int), cudaMemcpyHostToDevice, h->st));
    CK(cudaMemcpyAsync(&h->d.ctl->n_free, &n_free, sizeof(int), cudaMemcpyHostToDevice, h->st));
    CK(cudaStreamSynchronize(h->st));  // the host vectors above are temporaries
    return CFNEB_OK;
}

// Host mirrors of P / order / free slots after the device edited them (cfneb_step_adaptive).  Synchronises.
int sync_mirror(cfneb *h) {
    if (!h->mirror_dirty) return CFNEB_OK;
    Ctl c;
    std::vector<int> ord(h->d.S), fs(h->d.S);
    CK(cudaMemcpyAsync(&c, h->d.ctl, sizeof c, cudaMemcpyDeviceToHost, h->st));
    CK(cudaMemcpyAsync(ord.data(), h->d.order, sizeof(int) * h->d.S, cudaMemcpyDeviceToHost, h->st));
    CK(cudaMemcpyAsync(fs.data(), h->d.free_stack, sizeof(int) * h->d.S, cudaMemcpyDeviceToHost, h->st));
    CK(cudaStreamSynchronize(h->st));
    if (c.P < 3 || c.P > h->d.S || c.n_free < 0 || c.n_free > h->d.S) return CFNEB_ERANGE;
    h->P = c.P;
    h->order.assign(ord.begin(), ord.begin() + c.P);
    h->free_slots.assign(fs.begin(), fs.begin() + c.n_free);
    h->mirror_dirty = false;
    return CFNEB_OK;
}

// Reference cell h0 (A7), lam (A13) and the per-axis bin caps, from the two endpoint cells.
int set_reference_frame(cfneb *h, const double *cell_init, const double *cell_final) {
    Dev &d = h->d;
    memcpy(d.h0, cell_init, sizeof d.h0);  // A7: reference cell = cell of the initial endpoint
    inv3(d.h0, d.h0inv);
    // A13: lam = 0 selects Omega0^(1/3) N^(1/6); lam = 1 is the paper's equations literally
    d.lam = h->prm.cell_factor > 0.0 ? h->prm.cell_factor : cbrt(fabs(det3(cell_init))) * pow((double)d.N, 1.0 / 6.0);
    // per-axis bin caps from the larger endpoint cell, with headroom; product <= nbins_max
    double w0[3], w1[3];
    perp_widths(cell_init, w0);
    perp_widths(cell_final, w1);
    for (int a = 0; a < 3; ++a) {
        const double w = fmax(w0[a], w1[a]) * 1.5;
        d.nb_cap[a] = (int)floor(w / d.r_list);
        if (d.nb_cap[a] < 3) d.nb_cap[a] = 3;
    }
    while ((long long)d.nb_cap[0] * d.nb_cap[1] * d.nb_cap[2] > d.nbins_max) {
        int a = 0;
        if (d.nb_cap[1] > d.nb_cap[a]) a = 1;
        if (d.nb_cap[2] > d.nb_cap[a]) a = 2;
        if (d.nb_cap[a] <= 3) break;
        d.nb_cap[a] -= 1;
    }
    if ((long long)d.nb_cap[0] * d.nb_cap[1] * d.nb_cap[2] > d.nbins_max) return CFNEB_EINVAL;
    return CFNEB_OK;
}

int no_graph() {  // a failed cfneb_relax_endpoints(rebuild_band) leaves the handle without its iteration graph
    snprintf(g_cuda_err, sizeof g_cuda_err, "the handle has no iteration graph (an earlier cfneb_relax_endpoints failed while "
             "rebuilding the band); destroy it and create a new one");
    return CFNEB_ECUDA;
}

int capture_graph(cfneb *h) {
    CK(cudaStreamBeginCapture(h->st, cudaStreamCaptureModeRelaxed));
    enqueue_step(h, nullptr);
    cudaGraph_t g = nullptr;
    CK(cudaStreamEndCapture(h->st, &g));
    h->graph = g;
    size_t n_nodes = 0;
    CK(cudaGraphGetNodes(g, nullptr, &n_nodes));
    h->graph_nodes = (int)n_nodes;
    CK(cudaGraphInstantiate(&h->exec, g, 0));
    return CFNEB_OK;
}
}  // namespace

extern "C" {

void cfneb_default_params(cfneb_params *prm) {
    if (!prm) return;
    memset(prm, 0, sizeof *prm);
    prm->potential = CFNEB_POT_LJ_SF;
    prm->cell_mode = CFNEB_CELL_B;
    prm->climb = 1;
    prm->fire_nmin = 5;
    prm->max_neighbors = 160;
    prm->max_images = 16;
    prm->rebuild_every = 0;
    prm->pot[0] = 1.0; prm->pot[1] = 1.0; prm->pot[2] = 2.5;
    prm->k_spring = 1.0;
    prm->cell_factor = 1.0;
    prm->fire_dt0 = 0.1; prm->fire_dtmax = 1.0; prm->fire_maxstep = 0.2;
    prm->fire_finc = 1.1; prm->fire_fdec = 0.5; prm->fire_astart = 0.1; prm->fire_fa = 0.99;
    prm->skin = 0.3;
    prm->pressure = 0.0;
}

size_t cfneb_workspace_bytes(int32_t n_atoms, const cfneb_params *prm) {
    if (!valid_params(n_atoms, prm)) return 0;
    return carve(n_atoms, prm, nullptr, nullptr);
}

int cfneb_create(cfneb_t **out, int32_t n_atoms, const double *pos_init, const double *cell_init,
                 const double *pos_final, const double *cell_final, int32_t n_images, const double *path_or_null,
                 const cfneb_params *prm, void *dev_workspace, size_t ws_bytes, void *cuda_stream) {
    if (!out) return CFNEB_EINVAL;
    *out = nullptr;
    if (!valid_params(n_atoms, prm) || !pos_init || !cell_init || !pos_final || !cell_final || !dev_workspace)
        return CFNEB_EINVAL;
    if (n_images < 3) return CFNEB_EINVAL;
    if (n_images > prm->max_images) return CFNEB_ERANGE;
    if (reinterpret_cast<uintptr_t>(dev_workspace) & 255u) return CFNEB_EINVAL;
    if (ws_bytes < carve(n_atoms, prm, nullptr, nullptr)) return CFNEB_ENOMEM;
    const double vol0 = det3(cell_init), vol1 = det3(cell_final);
    if (!(fabs(vol0) > 0.0) || !(fabs(vol1) > 0.0) || !std::isfinite(vol0) || !std::isfinite(vol1)) return CFNEB_ECELL;

    cfneb *h = new (std::nothrow) cfneb();
    if (!h) return CFNEB_ENOMEM;
    h->prm = *prm;
    h->graph = nullptr;
    h->exec = nullptr;
    h->own_stream = false;
    h->interior_stale = false;
    h->mirror_dirty = false;
    h->st = static_cast<cudaStream_t>(cuda_stream);
    h->device = 0;
    h->st2 = nullptr;
    cudaGetDevice(&h->device);
#define CKH(call)                                  \
    do {                                           \
        int rc_ = (call);                          \
        if (rc_ != CFNEB_OK) { cfneb_destroy(h); return rc_; } \
    } while (0)
#define CKC(call)                                                                                      \
    do {                                                                                               \
        cudaError_t e_ = (call);                                                                       \
        if (e_ != cudaSuccess) {                                                                       \
            snprintf(g_cuda_err, sizeof g_cuda_err, "%s at %s:%d: %s", #call, __FILE__, __LINE__,     \
                     cudaGetErrorString(e_));                                                          \
            cfneb_destroy(h);                                                                          \
            return CFNEB_ECUDA;                                                                        \
        }                                                                                              \
    } while (0)
    if (!h->st) {
        CKC(cudaStreamCreate(&h->st));
        h->own_stream = true;
    }
    Dev &d = h->d;
    carve(n_atoms, prm, dev_workspace, &d);
    plan_stream_grids(d);
    d.potential = prm->potential;
    d.cell_mode = prm->cell_mode;
    d.climb = prm->climb ? 1 : 0;
    d.fire_nmin = prm->fire_nmin;
    d.rebuild_every = prm->rebuild_every;
    memcpy(d.pot, prm->pot, sizeof d.pot);
    d.k_spring = prm->k_spring;
    d.dt0 = prm->fire_dt0; d.dtmax = prm->fire_dtmax; d.maxstep = prm->fire_maxstep;
    d.finc = prm->fire_finc; d.fdec = prm->fire_fdec; d.astart = prm->fire_astart; d.fa = prm->fire_fa;
    d.skin = prm->skin;
    d.pressure = prm->pressure;
    d.r_cut = cutoff_of(prm);
    d.r_list = d.r_cut + d.skin;
    d.edge_b0 = prm->potential == CFNEB_POT_NEP
                    ? (int)floor(prm->pot[1] * prm->pot[1] / (d.r_cut * d.r_cut) * kInnerBuckets) : 0;
    prepare_potential(d);
    if (d.potential == CFNEB_POT_NEP) CKC(prepare_nep_kernels());
    if (set_reference_frame(h, cell_init, cell_final) != CFNEB_OK) { cfneb_destroy(h); return CFNEB_EINVAL; }
    h->P = n_images;
    h->order.resize(n_images);
    for (int p = 0; p < n_images; ++p) h->order[p] = p;
    for (int s = d.S - 1; s >= n_images; --s) h->free_slots.push_back(s);

    CKC(cudaMemsetAsync(dev_workspace, 0, carve(n_atoms, prm, nullptr, nullptr), h->st));
    Ctl c0;
    memset(&c0, 0, sizeof c0);
    c0.P = n_images;
    c0.first = 1;
    c0.pstar = -1;
    c0.dt = d.dt0;
    c0.alpha = d.astart;
    CKC(cudaMemcpyAsync(d.ctl, &c0, sizeof c0, cudaMemcpyHostToDevice, h->st));
    if (d.potential == CFNEB_POT_DNN) {  // network weights: the SplitMix64 stream of include/cfneb.h
        const int K = (int)d.pot[1], D = K + (int)d.pot[2] * (int)d.pot[3], H = (int)d.pot[4];
        double w[kDnWeights] = {0.0};
        uint64_t state = (uint64_t)d.pot[5];
        for (int t = 0; t < H * D + 2 * H; ++t) {
            uint64_t z = (state += 0x9E3779B97F4A7C15ull);
            z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
            z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
            z ^= z >> 31;
            const double u = 2.0 * ldexp((double)(z >> 11), -53) - 1.0;
            w[t] = t < H * D ? u * (t % D < K ? 0.3 / 8.0 : 0.3 / 40.0) : t < H * D + H ? 0.5 * u : u;
        }
        CKC(cudaMemcpyAsync(d.dn_w, w, sizeof w, cudaMemcpyHostToDevice, h->st));
        CKC(cudaStreamSynchronize(h->st));  // `w` is a temporary
    }
    CKH(upload_order(h));
    {
        std::vector<int> perm;
        spatial_order(n_atoms, pos_init, cell_init, d.r_list, perm);
        perm.resize(d.Npad, 0);
        CKC(cudaMemcpyAsync(d.perm, perm.data(), sizeof(int) * d.Npad, cudaMemcpyHostToDevice, h->st));
        CKC(cudaStreamSynchronize(h->st));  // `perm` is a temporary
        if (d.potential == CFNEB_POT_NEP) {  // atom types in storage order; the weight stream of include/cfneb.h
            const int T = (int)d.pot[8];
            std::vector<int> ty(d.Npad, 0);
            for (int i = 0; i < n_atoms; ++i) {
                const int t = prm->types ? prm->types[perm[i]] : 0;
                if (t < 0 || t >= T) { cfneb_destroy(h); return CFNEB_EINVAL; }
                ty[i] = t;
            }
            std::vector<double> w(nep_weight_count(d.pot));
            nep_fill_weights(d.pot, w.data());
            CKC(cudaMemcpyAsync(d.types, ty.data(), sizeof(int) * d.Npad, cudaMemcpyHostToDevice, h->st));
            CKC(cudaMemcpyAsync(d.dn_w, w.data(), sizeof(double) * w.size(), cudaMemcpyHostToDevice, h->st));
            CKC(cudaStreamSynchronize(h->st));  // temporaries
        }
    }

    // stage the host inputs: pos [n][N][3] then cells [n][9]
    const size_t N3 = (size_t)n_atoms * 3;
    const int n_in = path_or_null ? n_images : 2;
    std::vector<double> stage((size_t)n_in * (N3 + 9));
    double *spos = stage.data(), *scell = stage.data() + (size_t)n_in * N3;
    memcpy(spos, pos_init, N3 * sizeof(double));
    memcpy(scell, cell_init, 9 * sizeof(double));
    memcpy(spos + (size_t)(n_in - 1) * N3, pos_final, N3 * sizeof(double));
    memcpy(scell + (size_t)(n_in - 1) * 9, cell_final, 9 * sizeof(double));
    if (path_or_null)
        for (int q = 0; q < n_images - 2; ++q) {
            const double *blk = path_or_null + (size_t)q * (N3 + 9);
            memcpy(spos + (size_t)(q + 1) * N3, blk, N3 * sizeof(double));
            memcpy(scell + (size_t)(q + 1) * 9, blk + N3, 9 * sizeof(double));
            const double v = det3(blk + N3);
            if (!(fabs(v) > 0.0) || !std::isfinite(v)) { cfneb_destroy(h); return CFNEB_ECELL; }
        }
    double *dstage = static_cast<double *>(d.scratch);
    CKC(cudaMemcpyAsync(dstage, stage.data(), stage.size() * sizeof(double), cudaMemcpyHostToDevice, h->st));
    const double *dpos = dstage, *dcell = dstage + (size_t)n_in * N3;
    if (path_or_null) {
        launch_input_map(d, dpos, dcell, 0, n_images, 0, h->st);
    } else {
        launch_input_map(d, dpos, dcell, 0, 1, 0, h->st);
        launch_input_map(d, dpos + N3, dcell + 9, n_images - 1, 1, 0, h->st);
        launch_interpolate(d, n_images, h->st);
    }
    CKC(cudaStreamSynchronize(h->st));  // `stage` is a temporary
    CKH(force_rebuild_all(h));
    enqueue_evaluate_all(h);
    int rc = sync_status(h);
    if (rc) { cfneb_destroy(h); return rc; }
    CKH(capture_graph(h));
    *out = h;
    return CFNEB_OK;
#undef CKH
#undef CKC
}

int cfneb_step(cfneb_t *h, int32_t n_steps) {
    DeviceGuard dev_guard(h);
    if (!h || n_steps < 0) return CFNEB_EINVAL;
    if (!h->exec) return no_graph();
    if (n_steps > 0) h->interior_stale = false;
    for (int k = 0; k < n_steps; ++k) CK(cudaGraphLaunch(h->exec, h->st));
    return CFNEB_OK;
}

int cfneb_step_adaptive(cfneb_t *h, int32_t n_steps, int32_t adapt_every, double d_insert, double d_delete) {
    DeviceGuard dev_guard(h);
    if (!h || n_steps < 0 || adapt_every < 1) return CFNEB_EINVAL;
    if (!h->exec) return no_graph();
    if (n_steps > 0) h->interior_stale = false;
    for (int k = 1; k <= n_steps; ++k) {
        CK(cudaGraphLaunch(h->exec, h->st));
        if (k % adapt_every == 0) {
            launch_adapt_device(h->d, d_insert, d_delete, h->st);
            h->mirror_dirty = true;
        }
    }
    CK(cudaGetLastError());
    return CFNEB_OK;
}

int cfneb_step_timed(cfneb_t *h, int32_t n_steps, double *kernel_ms) {
    DeviceGuard dev_guard(h);
    if (!h || n_steps < 0 || !kernel_ms) return CFNEB_EINVAL;
    if (n_steps > 0) h->interior_stale = false;
    // one event set per step, read back after the last step: no host synchronisation between steps
    const int per = CFNEB_NKERNELS + 1;
    std::vector<cudaEvent_t> ev((size_t)n_steps * per, nullptr);
    int rc = CFNEB_OK;
    for (size_t k = 0; k < ev.size() && rc == CFNEB_OK; ++k)
        if (cudaEventCreate(&ev[k]) != cudaSuccess) rc = CFNEB_ECUDA;
    if (rc == CFNEB_OK) {
        for (int k = 0; k < n_steps; ++k) enqueue_step(h, ev.data() + (size_t)k * per);
        rc = sync_status(h);
    }
    if (rc == CFNEB_OK)
        for (int k = 0; k < n_steps; ++k)
            for (int c = 0; c < CFNEB_NKERNELS; ++c) {
                float ms = 0.f;
                if (cudaEventElapsedTime(&ms, ev[(size_t)k * per + c], ev[(size_t)k * per + c + 1]) != cudaSuccess) rc = CFNEB_ECUDA;
                kernel_ms[c] += (double)ms;
            }
    for (cudaEvent_t e : ev)
        if (e) cudaEventDestroy(e);
    if (rc == CFNEB_ECUDA) snprintf(g_cuda_err, sizeof g_cuda_err, "cfneb_step_timed: %s", cudaGetErrorString(cudaGetLastError()));
    return rc;
}

int cfneb_insert_image(cfneb_t *h, int32_t after) {
    DeviceGuard dev_guard(h);
    if (!h) return CFNEB_EINVAL;
    { int rc_m = sync_mirror(h); if (rc_m) return rc_m; }
    if (after < 0 || after > h->P - 2) return CFNEB_ERANGE;
    if (h->P >= h->d.S || h->free_slots.empty()) return CFNEB_ERANGE;
    int pstar = -1;
    CK(cudaMemcpyAsync(&pstar, &h->d.ctl->pstar, sizeof(int), cudaMemcpyDeviceToHost, h->st));
    CK(cudaStreamSynchronize(h->st));
    if (pstar > after) {  // keep the reported climbing index on the same image until the next step
        pstar += 1;
        CK(cudaMemcpyAsync(&h->d.ctl->pstar, &pstar, sizeof(int), cudaMemcpyHostToDevice, h->st));
        CK(cudaStreamSynchronize(h->st));
    }
    const int sn = h->free_slots.back();
    h->free_slots.pop_back();
    launch_midpoint(h->d, h->order[after], h->order[after + 1], sn, h->st);
    h->order.insert(h->order.begin() + after + 1, sn);
    h->P += 1;
    int rc = upload_order(h);
    if (rc) return rc;
    launch_reset_fire(h->d, h->st);
    CK(cudaGetLastError());
    return CFNEB_OK;
}

int cfneb_delete_image(cfneb_t *h, int32_t index) {
    DeviceGuard dev_guard(h);
    if (!h) return CFNEB_EINVAL;
    { int rc_m = sync_mirror(h); if (rc_m) return rc_m; }
    if (index < 1 || index > h->P - 2 || h->P <= 3) return CFNEB_ERANGE;
    int pstar = -1;
    CK(cudaMemcpyAsync(&pstar, &h->d.ctl->pstar, sizeof(int), cudaMemcpyDeviceToHost, h->st));
    CK(cudaStreamSynchronize(h->st));
    if (index == pstar) return CFNEB_ERANGE;
    h->free_slots.push_back(h->order[index]);
    h->order.erase(h->order.begin() + index);
    h->P -= 1;
    if (pstar > index) {  // keep the reported climbing index on the same image until the next step
        pstar -= 1;
        CK(cudaMemcpyAsync(&h->d.ctl->pstar, &pstar, sizeof(int), cudaMemcpyHostToDevice, h->st));
        CK(cudaStreamSynchronize(h->st));
    }
    int rc = upload_order(h);
    if (rc) return rc;
    launch_reset_fire(h->d, h->st);
    CK(cudaGetLastError());
    return CFNEB_OK;
}

int cfneb_get_segment_lengths(cfneb_t *h, double *dl) {
    DeviceGuard dev_guard(h);
    if (!h || !dl) return CFNEB_EINVAL;
    { int rc_m = sync_mirror(h); if (rc_m) return rc_m; }
    double *dev = static_cast<double *>(h->d.scratch);
    launch_segment_lengths(h->d, dev, h->st);
    CK(cudaMemcpyAsync(dl, dev, sizeof(double) * (h->P - 1), cudaMemcpyDeviceToHost, h->st));
    return sync_status(h);
}

int cfneb_adapt(cfneb_t *h, double d_insert, double d_delete, int32_t *n_ins, int32_t *n_del) {
    DeviceGuard dev_guard(h);
    if (!h) return CFNEB_EINVAL;
    { int rc_m = sync_mirror(h); if (rc_m) return rc_m; }
    if (n_ins) *n_ins = 0;
    if (n_del) *n_del = 0;
    std::vector<double> dl(h->d.S);
    int rc = cfneb_get_segment_lengths(h, dl.data());
    if (rc) return rc;
    int pstar = -1;
    CK(cudaMemcpyAsync(&pstar, &h->d.ctl->pstar, sizeof(int), cudaMemcpyDeviceToHost, h->st));
    CK(cudaStreamSynchronize(h->st));
    // (i) delete the interior, non-climbing image q minimising d_{q-1} + d_q if below d_delete and P > 3
    if (h->P > 3) {
        int best = -1;
        double bs = 0.0;
        for (int q = 1; q <= h->P - 2; ++q) {
            if (q == pstar) continue;
            const double s = dl[q - 1] + dl[q];
            if (best < 0 || s < bs) { best = q; bs = s; }
        }
        if (best > 0 && bs < d_delete) {
            rc = cfneb_delete_image(h, best);
            if (rc) return rc;
            if (n_del) *n_del = 1;
            rc = cfneb_get_segment_lengths(h, dl.data());
            if (rc) return rc;
        }
    }
    // (ii) insert at the midpoint of the longest segment if above d_insert and P < max_images
    int q = 0;
    for (int k = 1; k <= h->P - 2; ++k)
        if (dl[k] > dl[q]) q = k;
    if (dl[q] > d_insert && h->P < h->d.S) {
        rc = cfneb_insert_image(h, q);
        if (rc) return rc;
        if (n_ins) *n_ins = 1;
    }
    return sync_status(h);
}

int cfneb_reparametrize(cfneb_t *h, int32_t hold_climbing) {
    DeviceGuard dev_guard(h);
    if (!h) return CFNEB_EINVAL;
    launch_reparametrize(h->d, hold_climbing ? 1 : 0, h->st);
    h->interior_stale = true;
    CK(cudaGetLastError());
    return CFNEB_OK;
}

int cfneb_relax_endpoints(cfneb_t *h, double fmax_tol, int32_t max_steps, int32_t rebuild_band, int32_t *steps_done,
                          double *fmax_out, double *energy_out) {
    DeviceGuard dev_guard(h);
    if (!h || !(fmax_tol >= 0.0) || max_steps < 0) return CFNEB_EINVAL;
    { int rc_m = sync_mirror(h); if (rc_m) return rc_m; }
    const Dev &d = h->d;
    cudaStream_t st = h->st;
    launch_relax_init(d, st);
    RelaxState rs[2];
    memset(rs, 0, sizeof rs);
    int done = 0;
    const int chunk = 20;
    while (done < max_steps) {
        const int n = std::min(chunk, max_steps - done);
        for (int k = 0; k < n; ++k) {
            launch_cell_prep(d, kEndpointsOnly, MODE_STEP, st);
            launch_neighbor_build(d, kEndpointsOnly, st);
            launch_force(d, kEndpointsOnly, st);
            launch_finalize(d, kEndpointsOnly, st);
            launch_relax_step(d, fmax_tol, st);
        }
        done += n;
        CK(cudaMemcpyAsync(rs, d.relax, sizeof rs, cudaMemcpyDeviceToHost, st));
        int rc = sync_status(h);
        if (rc) return rc;
        if (rs[0].frozen && rs[1].frozen) break;
    }
    // energies / forces of the final endpoint states (the last update may have moved them)
    launch_cell_prep(d, kEndpointsOnly, MODE_STEP, st);
    launch_neighbor_build(d, kEndpointsOnly, st);
    launch_force(d, kEndpointsOnly, st);
    launch_finalize(d, kEndpointsOnly, st);
    launch_relax_step(d, 1e300, st);  // tol = inf: measures fmax and E, freezes, moves nothing
    CK(cudaMemcpyAsync(rs, d.relax, sizeof rs, cudaMemcpyDeviceToHost, st));
    int rc = sync_status(h);
    if (rc) return rc;
    for (int e = 0; e < 2; ++e) {
        if (steps_done) steps_done[e] = rs[e].steps;
        if (fmax_out) fmax_out[e] = rs[e].fmax;
        if (energy_out) energy_out[e] = rs[e].E;
    }
    launch_relax_init(d, st);  // endpoint velocities back to zero
    if (!rebuild_band) {
        launch_reset_fire(d, st);
        return sync_status(h);
    }
    // rebuild the band from the relaxed endpoints exactly as cfneb_create(endpoints only) would:
    // h0 := relaxed cell of image 0 (A7), lam (A13), interior images linear in X, fresh lists, new graph
    const size_t N3 = (size_t)d.N * 3, P = h->P;
    double *dpos = static_cast<double *>(d.scratch), *dcell = dpos + P * N3, *dE = dcell + P * 9;
    launch_cell_prep(d, 0, MODE_GEOMETRY_ONLY, st);
    launch_export_path(d, dpos, dcell, dE, st);
    double cell0[9], cell1[9];
    CK(cudaMemcpyAsync(cell0, dcell, sizeof cell0, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(cell1, dcell + (P - 1) * 9, sizeof cell1, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (h->exec) { cudaGraphExecDestroy(h->exec); h->exec = nullptr; }
    if (h->graph) { cudaGraphDestroy(h->graph); h->graph = nullptr; }
    rc = set_reference_frame(h, cell0, cell1);
    if (rc) return rc;
    // the exported Cartesian endpoints sit in the first half of the scratch area; input_map reads them there
    launch_input_map(h->d, dpos, dcell, 0, 1, 0, st);
    launch_input_map(h->d, dpos + (P - 1) * N3, dcell + (P - 1) * 9, (int)P - 1, 1, 0, st);
    launch_interpolate(h->d, (int)P, st);
    launch_reset_fire(h->d, st);
    rc = force_rebuild_all(h);
    if (rc) return rc;
    enqueue_evaluate_all(h);
    rc = sync_status(h);
    if (rc) return rc;
    return capture_graph(h);
}

int cfneb_get_path(cfneb_t *h, int32_t *n_images, double *pos, double *cells, double *energies) {
    DeviceGuard dev_guard(h);
    if (!h) return CFNEB_EINVAL;
    { int rc_m = sync_mirror(h); if (rc_m) return rc_m; }
    const Dev &d = h->d;
    const size_t N3 = (size_t)d.N * 3, P = h->P;
    double *dpos = static_cast<double *>(d.scratch), *dcell = dpos + P * N3, *dE = dcell + P * 9;
    if (energies && h->interior_stale) {  // the path was replaced and never evaluated: do it now
        enqueue_evaluate_all(h);
        h->interior_stale = false;
    }
    launch_cell_prep(d, 0, MODE_GEOMETRY_ONLY, h->st);
    launch_export_path(d, dpos, dcell, dE, h->st);
    if (pos) CK(cudaMemcpyAsync(pos, dpos, P * N3 * sizeof(double), cudaMemcpyDeviceToHost, h->st));
    if (cells) CK(cudaMemcpyAsync(cells, dcell, P * 9 * sizeof(double), cudaMemcpyDeviceToHost, h->st));
    if (energies) CK(cudaMemcpyAsync(energies, dE, P * sizeof(double), cudaMemcpyDeviceToHost, h->st));
    if (n_images) *n_images = h->P;
    return sync_status(h);
}

int cfneb_set_path(cfneb_t *h, const double *pos, const double *cells) {
    DeviceGuard dev_guard(h);
    if (!h || !pos || !cells) return CFNEB_EINVAL;
    { int rc_m = sync_mirror(h); if (rc_m) return rc_m; }
    const Dev &d = h->d;
    const size_t N3 = (size_t)d.N * 3, P = h->P;
    double *dpos = static_cast<double *>(d.scratch), *dcell = dpos + P * N3;
    CK(cudaMemcpyAsync(dpos, pos, P * N3 * sizeof(double), cudaMemcpyHostToDevice, h->st));
    CK(cudaMemcpyAsync(dcell, cells, P * 9 * sizeof(double), cudaMemcpyHostToDevice, h->st));
    // The neighbour lists are kept: input_map records how far the new coordinates are from the stored ones, and the
    // K0 pass over ALL images that follows adds that to every image's displacement bound, rebuilds the lists that
    // left their skin and measures the exact displacement of the new path from the build-time coordinates -- so the
    // bound never has to cover more than one replacement (a checkpoint restore or a host-side edit of a few images
    // costs no rebuild of the others).
    launch_input_map(d, dpos, dcell, 0, h->P, 1, h->st);
    launch_reset_fire(d, h->st);
    launch_cell_prep(d, 0, MODE_STEP, h->st);
    launch_neighbor_build(d, 0, h->st);
    // endpoint energies now; the interior is evaluated by the next cfneb_step / cfneb_get_forces, or on demand by
    // cfneb_get_path (interior_stale)
    launch_force(d, kEndpointsOnly, h->st);
    launch_finalize(d, kEndpointsOnly, h->st);
    h->interior_stale = true;
    return sync_status(h);
}

int cfneb_get_state(cfneb_t *h, double *X, double *v) {
    DeviceGuard dev_guard(h);
    if (!h) return CFNEB_EINVAL;
    { int rc_m = sync_mirror(h); if (rc_m) return rc_m; }
    const Dev &d = h->d;
    const size_t n = (size_t)h->P * (d.N + 3) * 3;
    double *dX = static_cast<double *>(d.scratch), *dv = dX + n;
    launch_export_state(d, dX, dv, h->st);
    if (X) CK(cudaMemcpyAsync(X, dX, n * sizeof(double), cudaMemcpyDeviceToHost, h->st));
    if (v) CK(cudaMemcpyAsync(v, dv, n * sizeof(double), cudaMemcpyDeviceToHost, h->st));
    return sync_status(h);
}

int cfneb_get_checkpoint(cfneb_t *h, double *X, double *v, double *X_list, double *list_aux, cfneb_fire_state *fire) {
    DeviceGuard dev_guard(h);
    if (!h) return CFNEB_EINVAL;
    int rc = (X || v) ? cfneb_get_state(h, X, v) : sync_mirror(h);
    if (rc) return rc;
    const Dev &d = h->d;
    const size_t n = (size_t)h->P * (d.N + 3) * 3;
    if (X_list || list_aux) {
        double *dX = static_cast<double *>(d.scratch), *daux = dX + n;
        launch_export_list_state(d, dX, daux, h->st);
        if (X_list) CK(cudaMemcpyAsync(X_list, dX, n * sizeof(double), cudaMemcpyDeviceToHost, h->st));
        if (list_aux) CK(cudaMemcpyAsync(list_aux, daux, (size_t)h->P * 4 * sizeof(double), cudaMemcpyDeviceToHost, h->st));
    }
    if (fire) {
        Ctl c;
        CK(cudaMemcpyAsync(&c, d.ctl, sizeof c, cudaMemcpyDeviceToHost, h->st));
        CK(cudaStreamSynchronize(h->st));
        fire->dt = c.dt;
        fire->alpha = c.alpha;
        fire->steps = (int64_t)c.steps;
        fire->n_pos = c.n_pos;
        fire->first = c.first;
    }
    return sync_status(h);
}

int cfneb_set_state(cfneb_t *h, const double *X, const double *v, const double *X_list, const double *list_aux,
                    const cfneb_fire_state *fire) {
    DeviceGuard dev_guard(h);
    if (!h || !X || (X_list && !list_aux)) return CFNEB_EINVAL;
    if (fire && (!(fire->dt > 0.0) || !(fire->alpha >= 0.0) || fire->n_pos < 0 || fire->steps < 0)) return CFNEB_EINVAL;
    { int rc_m = sync_mirror(h); if (rc_m) return rc_m; }
    const Dev &d = h->d;
    cudaStream_t st = h->st;
    const size_t n = (size_t)h->P * (d.N + 3) * 3;
    double *dX = static_cast<double *>(d.scratch), *dv = dX + n;
    int rc;
    if (X_list) {  // replay the list builds: lists at X_list, then the coordinates proper
        CK(cudaMemcpyAsync(dX, X_list, n * sizeof(double), cudaMemcpyHostToDevice, st));
        // an image whose rebuild was pending at the checkpoint (list_aux[4p+3] < 0: inserted and not yet stepped) has no
        // build coordinates worth replaying -- an unused slot exports zeros, which are not a cell: its list is built at X
        // here and, the flag restored below, again by the next K0, exactly as the uninterrupted band does
        const size_t row = (size_t)(d.N + 3) * 3;
        for (int p = 0; p < h->P; ++p)
            if (list_aux[4 * p + 3] < 0.0)
                CK(cudaMemcpyAsync(dX + p * row, X + p * row, row * sizeof(double), cudaMemcpyHostToDevice, st));
        launch_import_state(d, dX, nullptr, 0, 0, h->P, st);
        CK(cudaStreamSynchronize(st));
        rc = force_rebuild_all(h);
        if (rc) return rc;
        launch_cell_prep(d, 0, MODE_STEP, st);
        launch_neighbor_build(d, 0, st);
    }
    CK(cudaMemcpyAsync(dX, X, n * sizeof(double), cudaMemcpyHostToDevice, st));
    if (v && fire) CK(cudaMemcpyAsync(dv, v, n * sizeof(double), cudaMemcpyHostToDevice, st));
    // without X_list the neighbour lists are kept: the distance of the new coordinates from the stored ones goes into
    // each image's staleness bound (as in cfneb_set_path), so a state that is the stored one -- the host round trip of a
    // running band -- rebuilds nothing and continues bit for bit
    launch_import_state(d, dX, (v && fire) ? dv : nullptr, X_list ? 0 : 1, 0, h->P, st);
    if (!(v && fire)) launch_reset_fire(d, st);  // no velocities, or no FIRE state to go with them: a restart
    CK(cudaStreamSynchronize(st));  // dX / dv are reused below
    double *daux = dX;
    if (X_list) CK(cudaMemcpyAsync(daux, list_aux, (size_t)h->P * 4 * sizeof(double), cudaMemcpyHostToDevice, st));
    launch_import_aux(d, daux, X_list ? 1 : 0, fire ? 1 : 0, fire ? fire->dt : 0.0, fire ? fire->alpha : 0.0,
                      fire ? fire->n_pos : 0, fire ? (fire->first ? 1 : 0) : 1,
                      fire ? (unsigned long long)fire->steps : 0ull, st);
    // endpoint energies at the restored coordinates (their lists: replayed above, or fresh)
    launch_cell_prep(d, kEndpointsOnly, MODE_STEP, st);
    launch_neighbor_build(d, kEndpointsOnly, st);
    launch_force(d, kEndpointsOnly, st);
    launch_finalize(d, kEndpointsOnly, st);
    h->interior_stale = true;
    return sync_status(h);
}

int cfneb_step_hosted(cfneb_t *h, double *X, double *v, cfneb_fire_state *fire, int32_t n_blocks) {
    DeviceGuard dev_guard(h);
    if (!h || !X || n_blocks < 0) return CFNEB_EINVAL;  // v, fire: optional (nullptr = that part of the state stays resident)
    if (fire && (!(fire->dt > 0.0) || !(fire->alpha >= 0.0) || fire->n_pos < 0 || fire->steps < 0)) return CFNEB_EINVAL;
    { int rc_m = sync_mirror(h); if (rc_m) return rc_m; }
    const Dev &d = h->d;
    cudaStream_t st = h->st;
    const int P = h->P;
    if (P >= 4096) return CFNEB_ERANGE;  // image_block() packs first and count into 12 bits each
    if (n_blocks == 0) n_blocks = 10;
    if (n_blocks > P) n_blocks = P;
    if (!h->st2) CK(cudaStreamCreateWithFlags(&h->st2, cudaStreamNonBlocking));
    while ((int)h->ev_blocks.size() < n_blocks + 1) {
        cudaEvent_t e;
        CK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        h->ev_blocks.push_back(e);
    }
    const size_t row = (size_t)(d.N + 3) * 3, n = (size_t)P * row;
    double *dX = static_cast<double *>(d.scratch), *dv = dX + n;
    // the copy stream starts after everything enqueued on the handle's stream so far (the staging area may be in use)
    CK(cudaEventRecord(h->ev_blocks[n_blocks], st));
    CK(cudaStreamWaitEvent(h->st2, h->ev_blocks[n_blocks], 0));
    if (fire)
        launch_import_aux(d, nullptr, 0, 1, fire->dt, fire->alpha, fire->n_pos, fire->first ? 1 : 0, (unsigned long long)fire->steps, st);
    h->interior_stale = false;
    for (int b = 0; b < n_blocks; ++b) {
        const int a = (int)((long long)P * b / n_blocks), e = (int)((long long)P * (b + 1) / n_blocks), cnt = e - a;
        if (cnt <= 0) continue;
        CK(cudaMemcpyAsync(dX + a * row, X + a * row, cnt * row * sizeof(double), cudaMemcpyHostToDevice, h->st2));
        if (v) CK(cudaMemcpyAsync(dv + a * row, v + a * row, cnt * row * sizeof(double), cudaMemcpyHostToDevice, h->st2));
        CK(cudaEventRecord(h->ev_blocks[b], h->st2));
        CK(cudaStreamWaitEvent(st, h->ev_blocks[b], 0));
        // K0-K2 of an image need only that image's coordinates: the block is evaluated while the next ones arrive
        launch_import_state(d, dX, v ? dv : nullptr, 1, a, cnt, st);
        const int sel = image_block(a, cnt);
        launch_cell_prep(d, sel, MODE_STEP, st);
        launch_neighbor_build(d, sel, st);
        launch_force(d, sel, st);
        launch_finalize(d, sel, st);
    }
    // the endpoints as cfneb_set_state evaluates them (their energies enter the tangents of images 1 and P - 2)
    launch_cell_prep(d, kEndpointsOnly, MODE_STEP, st);
    launch_neighbor_build(d, kEndpointsOnly, st);
    launch_force(d, kEndpointsOnly, st);
    launch_finalize(d, kEndpointsOnly, st);
    launch_reduce(d, st);
    launch_scalar(d, 0, st);
    launch_update(d, st);
    launch_export_state(d, dX, v ? dv : nullptr, st);
    CK(cudaMemcpyAsync(X, dX, n * sizeof(double), cudaMemcpyDeviceToHost, st));
    if (v) CK(cudaMemcpyAsync(v, dv, n * sizeof(double), cudaMemcpyDeviceToHost, st));
    Ctl c;
    CK(cudaMemcpyAsync(&c, d.ctl, sizeof c, cudaMemcpyDeviceToHost, st));
    int rc = sync_status(h);
    if (rc) return rc;
    if (fire) {
        fire->dt = c.dt;
        fire->alpha = c.alpha;
        fire->steps = (int64_t)c.steps;
        fire->n_pos = c.n_pos;
        fire->first = c.first;
    }
    return CFNEB_OK;
}

int cfneb_get_forces(cfneb_t *h, double *F, double *virial, double *f_neb, double *energies) {
    DeviceGuard dev_guard(h);
    if (!h) return CFNEB_EINVAL;
    { int rc_m = sync_mirror(h); if (rc_m) return rc_m; }
    const Dev &d = h->d;
    const size_t N3 = (size_t)d.N * 3, P = h->P;
    h->interior_stale = false;
    launch_cell_prep(d, 1, MODE_STEP, h->st);
    launch_neighbor_build(d, 1, h->st);
    launch_force(d, 1, h->st);
    launch_finalize(d, 1, h->st);
    launch_reduce(d, h->st);
    launch_scalar(d, 1, h->st);
    launch_materialize_fneb(d, h->st);
    double *dF = static_cast<double *>(d.scratch), *dV = dF + P * N3, *dE = dV + P * 9;
    launch_export_forces(d, dF, dV, dE, h->st);
    if (F) CK(cudaMemcpyAsync(F, dF, P * N3 * sizeof(double), cudaMemcpyDeviceToHost, h->st));
    if (virial) CK(cudaMemcpyAsync(virial, dV, P * 9 * sizeof(double), cudaMemcpyDeviceToHost, h->st));
    if (energies) CK(cudaMemcpyAsync(energies, dE, P * sizeof(double), cudaMemcpyDeviceToHost, h->st));
    if (f_neb)
        CK(cudaMemcpyAsync(f_neb, d.fneb, P * (size_t)(d.N + 3) * 3 * sizeof(double), cudaMemcpyDeviceToHost, h->st));
    return sync_status(h);
}

int cfneb_get_dots(cfneb_t *h, double *dots, double *coef, double *G) {
    DeviceGuard dev_guard(h);
    if (!h) return CFNEB_EINVAL;
    { int rc_m = sync_mirror(h); if (rc_m) return rc_m; }
    const Dev &d = h->d;
    const size_t P = h->P;
    h->interior_stale = false;
    launch_cell_prep(d, 1, MODE_STEP, h->st);
    launch_neighbor_build(d, 1, h->st);
    launch_force(d, 1, h->st);
    launch_finalize(d, 1, h->st);
    launch_reduce(d, h->st);
    launch_scalar(d, 1, h->st);
    launch_materialize_gen_force(d, h->st);
    double *dD = static_cast<double *>(d.scratch), *dC = dD + P * kNDots;
    launch_export_dots(d, dD, dC, h->st);
    if (dots) CK(cudaMemcpyAsync(dots, dD, P * kNDots * sizeof(double), cudaMemcpyDeviceToHost, h->st));
    if (coef) CK(cudaMemcpyAsync(coef, dC, P * 4 * sizeof(double), cudaMemcpyDeviceToHost, h->st));
    if (G) CK(cudaMemcpyAsync(G, d.fneb, P * (size_t)(d.N + 3) * 3 * sizeof(double), cudaMemcpyDeviceToHost, h->st));
    return sync_status(h);
}

int cfneb_get_neighbors(cfneb_t *h, int32_t image, int32_t *count, int32_t *list, int32_t *shift) {
    DeviceGuard dev_guard(h);
    if (!h) return CFNEB_EINVAL;
    { int rc_m = sync_mirror(h); if (rc_m) return rc_m; }
    if (image < 0 || image >= h->P) return CFNEB_ERANGE;
    const Dev &d = h->d;
    const int slot = h->order[image];
    const int one = 1;
    CK(cudaMemcpyAsync(&d.geom[slot].force_rebuild, &one, sizeof(int), cudaMemcpyHostToDevice, h->st));
    launch_cell_prep(d, 0, MODE_STEP, h->st);
    launch_neighbor_build(d, 0, h->st);
    const size_t n = (size_t)d.N * d.cap_user;
    int *dcount = static_cast<int *>(d.scratch), *dlist = dcount + ((d.N + 63) / 64) * 64, *dshift = dlist + n;
    launch_unpack_neighbors(d, slot, dcount, dlist, dshift, h->st);
    if (count) CK(cudaMemcpyAsync(count, dcount, sizeof(int) * d.N, cudaMemcpyDeviceToHost, h->st));
    if (list) CK(cudaMemcpyAsync(list, dlist, sizeof(int) * n, cudaMemcpyDeviceToHost, h->st));
    if (shift) CK(cudaMemcpyAsync(shift, dshift, sizeof(int) * 3 * n, cudaMemcpyDeviceToHost, h->st));
    return sync_status(h);
}

int cfneb_get_status(cfneb_t *h, cfneb_status *out) {
    DeviceGuard dev_guard(h);
    if (!h || !out) return CFNEB_EINVAL;
    Ctl c;
    CK(cudaMemcpyAsync(&c, h->d.ctl, sizeof c, cudaMemcpyDeviceToHost, h->st));
    CK(cudaStreamSynchronize(h->st));
    memset(out, 0, sizeof *out);
    out->steps = (int64_t)c.steps;
    out->rebuilds = (int64_t)c.rebuilds;
    out->n_images = c.P;
    out->climb_index = c.pstar;
    out->error = c.error;
    out->n_pos = c.n_pos;
    out->max_neighbors_seen = c.max_nbr_seen;
    out->graph_kernel_nodes = h->graph_nodes;
    unsigned long long b = c.fmax_bits;
    double f2;
    memcpy(&f2, &b, sizeof f2);
    out->fmax = sqrt(f2);
    out->barrier = c.barrier;
    out->dt = c.dt;
    out->alpha = c.alpha;
    out->cell_factor = h->d.lam;
    out->path_length = c.path_length;
    CK(cudaGetLastError());
    return CFNEB_OK;
}

int cfneb_get_history(cfneb_t *h, int64_t first_step, int32_t n, cfneb_history_entry *out) {
    DeviceGuard dev_guard(h);
    if (!h || !out || n < 0) return CFNEB_EINVAL;
    if (n == 0) return CFNEB_OK;
    std::vector<double> ring((size_t)kHistLen * kHistFields);
    Ctl c;
    CK(cudaMemcpyAsync(ring.data(), h->d.hist, ring.size() * sizeof(double), cudaMemcpyDeviceToHost, h->st));
    CK(cudaMemcpyAsync(&c, h->d.ctl, sizeof c, cudaMemcpyDeviceToHost, h->st));
    CK(cudaStreamSynchronize(h->st));
    const int64_t last = (int64_t)c.steps;
    if (first_step < 1 || first_step + n - 1 > last || first_step + kHistLen <= last) return CFNEB_ERANGE;
    for (int32_t i = 0; i < n; ++i) {
        const int64_t s = first_step + i;  // the iteration after which status.steps == s; its row: index s - 1
        const double *row = ring.data() + (size_t)((s - 1) % kHistLen) * kHistFields;
        if (row[0] != (double)s) return CFNEB_ERANGE;  // not recorded (the counter was set by cfneb_set_state) or overwritten
        double f2 = row[1];
        if (s == last) {  // K6 of the last iteration left its maximum in the control block; no later K5 has filed it yet
            const unsigned long long b = c.fmax_bits;
            memcpy(&f2, &b, sizeof f2);
        }
        out[i].step = s;
        out[i].rebuilds = (int64_t)row[7];
        out[i].n_images = (int32_t)row[6];
        out[i].climb_index = (int32_t)row[3];
        out[i].fmax = sqrt(f2);
        out[i].barrier = row[2];
        out[i].dt = row[4];
        out[i].alpha = row[5];
    }
    return c.error;
}

void cfneb_destroy(cfneb_t *h) {
    if (!h) return;
    DeviceGuard dev_guard(h);
    if (h->st) cudaStreamSynchronize(h->st);
    if (h->exec) cudaGraphExecDestroy(h->exec);
    if (h->graph) cudaGraphDestroy(h->graph);
    for (cudaEvent_t e : h->ev_blocks) cudaEventDestroy(e);
    if (h->st2) cudaStreamDestroy(h->st2);
    if (h->own_stream && h->st) cudaStreamDestroy(h->st);
    delete h;
}

const char *cfneb_strerror(int code) {
    switch (code) {
        case CFNEB_OK: return "ok";
        case CFNEB_EINVAL: return "invalid argument (or zero tangent)";
        case CFNEB_ENOMEM: return "workspace too small";
        case CFNEB_ECUDA: return "CUDA runtime error";
        case CFNEB_ENEIGH_OVERFLOW: return "neighbour list overflow (raise max_neighbors)";
        case CFNEB_ECELL: return "cell not positive definite / singular / periodic shift out of range";
        case CFNEB_ENAN: return "NaN or Inf in energies or reductions";
        case CFNEB_ERANGE: return "image index out of range / endpoint or climbing image / band full";
        default: return "unknown error";
    }
}

const char *cfneb_last_cuda_error(void) { return g_cuda_err; }

int cfneb_util_fp64_peak(void *cuda_stream, double *tflops) {
    if (!tflops) return CFNEB_EINVAL;
    const double t = run_fp64_peak(static_cast<cudaStream_t>(cuda_stream));
    if (!(t > 0.0)) {
        snprintf(g_cuda_err, sizeof g_cuda_err, "fp64 peak kernel failed: %s", cudaGetErrorString(cudaGetLastError()));
        return CFNEB_ECUDA;
    }
    *tflops = t;
    return CFNEB_OK;
}

}  // extern "C"

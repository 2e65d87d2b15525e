/*
 * cfneb.h -- C ABI of the B200-native CFNEB hot path (arXiv:2510.16721).
 *
 * One handle = one nudged-elastic-band chain of P images of N atoms in a variable periodic cell,
 * resident in GPU memory.  `cfneb_step` runs the whole iteration of the paper's workflow
 * (PAPER.md "IMPLEMENTATION": cell filter -> force evaluation -> NEB iteration) for all
 * images at once, in fp64, as hand-written CUDA kernels for sm_100a captured in a CUDA graph;
 * `cfneb_adapt` / `cfneb_insert_image` / `cfneb_delete_image` are the image-distribution
 * adjustment of P:128.  Citations `P:n` are lines of the paper text, `O*`/`A*` are the
 * step definitions and readings of SURVEY.md §8(c) restated in DESIGN.md.
 *
 * Conventions (all arrays are plain row-major double / int32, HOST pointers unless stated):
 *   - row vectors; a cell is double[9], rows = lattice vectors h1,h2,h3, R = s h;
 *   - positions are Cartesian, double[N*3], never wrapped into the cell (A17);
 *   - generalized coordinates of an image: X = [R~ ; lam*B], (N+3) x 3, with R~ = R D^-1 (Eq. 10),
 *     D = h0^-1 h, B = D D^T (Eq. 15), h0 = cell of image 0 (A7), lam = cell_factor (A13);
 *   - generalized forces: [F D^T ; D^-T V D^-1 / lam] (Eq. 17, as printed, A9), V the virial of Eq. 8.
 *
 * Ownership: the caller owns every host buffer (the library copies in/out and never retains host
 * pointers) and owns the device workspace, which must stay alive and untouched until
 * cfneb_destroy.  The library allocates no device memory of its own after cfneb_create returns.
 *
 * Errors: every call returns 0 (CFNEB_OK) or a negative code; nothing throws or aborts across
 * the ABI.  Failures detected on the device (neighbour-list overflow, non-positive-definite B,
 * NaN) set a sticky error word that the next synchronising call returns and cfneb_get_status
 * reports; once set, further steps leave the state undefined.
 *
 * Threading: a handle must be used from one host thread at a time.  All device work is enqueued
 * on the CUDA stream given to cfneb_create.
 */
#ifndef CFNEB_H
#define CFNEB_H

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define CFNEB_API __attribute__((visibility("default")))
#else
#define CFNEB_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cfneb cfneb_t; /* opaque */

enum {
    CFNEB_OK = 0,
    CFNEB_EINVAL = -1,          /* bad argument (null pointer, n_images < 3, unknown enum, zero tangent ...) */
    CFNEB_ENOMEM = -2,          /* workspace too small */
    CFNEB_ECUDA = -3,           /* a CUDA runtime call failed; cfneb_last_cuda_error() has the text */
    CFNEB_ENEIGH_OVERFLOW = -4, /* an atom has more than max_neighbors neighbours within r_cut + skin */
    CFNEB_ECELL = -5,           /* B not positive definite / singular cell / periodic shift out of range */
    CFNEB_ENAN = -6,            /* NaN or Inf in energies or reductions */
    CFNEB_ERANGE = -7           /* bad image index, endpoint / climbing-image delete, more than max_images */
};

enum { CFNEB_POT_LJ_SF = 0, CFNEB_POT_FS_MORSE = 1, CFNEB_POT_SW = 2, CFNEB_POT_DNN = 3, CFNEB_POT_NEP = 4 };
enum { CFNEB_CELL_FIXED = 0, CFNEB_CELL_B = 1 /* Eq. 17, rotation-free (default) */, CFNEB_CELL_D = 2 /* Eq. 14 */ };

/*
 * Parameters (plain data, copied by cfneb_create).
 *   potential = CFNEB_POT_LJ_SF:   pot = {eps, sigma, r_c}: phi_SF(r) = phi(r) - phi(r_c) - (r - r_c) phi'(r_c)
 *   potential = CFNEB_POT_FS_MORSE: pot = {D, alpha, r0, beta, rho_r0, A, r_on, r_cut}:
 *       v(r) = D[e^{-2 alpha (r-r0)} - 2 e^{-alpha (r-r0)}] t(r), rho_i = sum_j e^{-beta (r - rho_r0)} t(r),
 *       U_i = 1/2 sum_j v + F(rho_i), F = -A sqrt(rho), t = cosine taper from r_on to r_cut (O3, A21).
 *   potential = CFNEB_POT_SW (Stillinger-Weber, three-body): pot = {eps, sigma, a, lambda, gamma, A, B, p, q}, r_c = a sigma:
 *       U_i = 1/2 sum_j A eps [B (sigma/r)^p - (sigma/r)^q] e^{sigma/(r - r_c)}
 *             + sum_{j<k} lambda eps (cos theta_jik + 1/3)^2 e^{gamma sigma/(r_ij - r_c)} e^{gamma sigma/(r_ik - r_c)},
 *       evaluated through the partial forces p^ij = dU_i/dr^ij of Eq. 5 (f^ij = p^ij - p^ji) and Eq. 8; at most 32
 *       neighbours inside r_c per atom (CFNEB_ENEIGH_OVERFLOW otherwise).
 *   potential = CFNEB_POT_DNN (descriptor network: the SHAPE of the paper's NEP potential, P:138 -- radial and
 *       angular descriptors of the environment into a one-hidden-layer network -- with seeded weights, because the
 *       trained ones are not available: a cost and data-flow stand-in, not a physical model):
 *       pot = {r_c, K, M, L, H, seed}, K, M <= 4 radial functions, L <= 3, H <= 8 neurons, D = K + M L <= 16:
 *       f_k(r) = 1/2 [T_k(x) + 1] fc(r), x = 2 (r/r_c - 1)^2 - 1, fc = 1/2 [1 + cos(pi r / r_c)] (T_k Chebyshev),
 *       q_k = sum_j f_k(r_ij) (k < K),  q_{K + n L + l - 1} = sum_j sum_k f_n(r_ij) f_n(r_ik) P_l(cos theta_jik)
 *       (n < M, l = 1..L, all ordered pairs j, k including j = k),  U_i = sum_mu W1_mu tanh(sum_d W0_{mu d} q_d - b0_mu).
 *       Weights: SplitMix64 stream from `seed`, u = (z >> 11) 2^-53, w = 2u - 1, in the order W0[mu][d] (scaled by
 *       0.3/8 for d < K, 0.3/40 otherwise), b0[mu] (scaled by 0.5), W1[mu].  Same two passes as CFNEB_POT_SW.
 *   potential = CFNEB_POT_NEP (the descriptor network widened to the shape and cost of the paper's force field proper,
 *       P:138 "NEP-trained force field"; seeded weights, a cost and data-flow stand-in):
 *       pot = {rc_r, rc_a, n_r, n_a, k_r, k_a, L, H, n_types, seed}: rc_a <= rc_r; n_r, n_a <= 8 radial descriptors /
 *       angular radial functions; k_r, k_a <= 12 basis functions; L <= 4; H <= 64 neurons; n_types <= 2 (`types`):
 *       f_k(r; rc) as above with its own cut-off,  g^R_n(r) = sum_{k<k_r} cR[I][J][n][k] f_k(r; rc_r),
 *       g^A_n(r) = sum_{k<k_a} cA[I][J][n][k] f_k(r; rc_a)   (I = type of atom i, J = type of the neighbour),
 *       q_n = sum_j g^R_n(r_ij) (n < n_r),  q_{n_r + n L + l - 1} = sum_j sum_k g^A_n(r_ij) g^A_n(r_ik) P_l(cos theta_jik)
 *       (n < n_a, l = 1..L, neighbours inside rc_a, all ordered pairs including j = k),
 *       U_i = sum_mu W1[I][mu] tanh(sum_d W0[I][mu][d] q_d - b0[I][mu]).
 *       Weights: one SplitMix64 stream from `seed`, w = 2u - 1, drawn in the order: for each type I: W0[I][mu][d]
 *       (scaled by 0.04 for d < n_r, 0.004 otherwise), b0[I][mu] (scaled by 0.5), W1[I][mu]; then cR[I][J][n][k];
 *       then cA[I][J][n][k].  The neighbour lists use rc_r.  Same two passes as CFNEB_POT_SW.
 *   types: CFNEB_POT_NEP only: HOST pointer to n_atoms atom types in [0, n_types), read by cfneb_create and not
 *       retained (NULL = all atoms of type 0).
 *   k_spring: uniform spring constant of Eq. 1 (A14).  climb: 1 = climbing image (ref [12]).
 *   cell_factor: lam of A13; 0 = auto (Omega0^(1/3) N^(1/6)); 1 = the paper's equations literally.
 *   fire_*: FIRE constants of O7 (one state for the whole band).
 *   skin: neighbour-list skin; lists hold pairs with r < r_cut + skin and are rebuilt on the device
 *         when the accumulated displacement bound exceeds skin, or every rebuild_every steps (0 = never
 *         by count).  max_neighbors: list capacity per atom.  max_images: capacity of the band.
 *   pressure: external hydrostatic pressure p in energy / length^3 (reading A25; the paper's graphite band is
 *         "under 40GPa").  The band then relaxes the enthalpy H = U + p Omega: every energy the library
 *         reports or uses (tangent, climbing image, barrier, cfneb_get_path / cfneb_get_forces) is H, and the
 *         virial is V - p Omega I (Eq. 2-3).  0 = none.
 */
typedef struct cfneb_params {
    int32_t potential;
    int32_t cell_mode;
    int32_t climb;
    int32_t fire_nmin;
    int32_t max_neighbors;
    int32_t max_images;
    int32_t rebuild_every;
    int32_t reserved0;
    double pot[12];
    double k_spring;
    double cell_factor;
    double fire_dt0, fire_dtmax, fire_maxstep, fire_finc, fire_fdec, fire_astart, fire_fa;
    double skin;
    double pressure;
    const int32_t *types;
} cfneb_params;

/* Snapshot written by cfneb_get_status (synchronises the stream). */
typedef struct cfneb_status {
    int64_t steps;          /* NEB iterations done since create */
    int64_t rebuilds;       /* per-image neighbour-list rebuilds done on the device */
    int32_t n_images;       /* current P */
    int32_t climb_index;    /* p* of the last step (path position), -1 if none */
    int32_t error;          /* sticky device error (0 or a negative CFNEB_E* code) */
    int32_t n_pos;          /* FIRE counter of consecutive power > 0 steps */
    int32_t max_neighbors_seen;
    int32_t graph_kernel_nodes; /* kernel launches of one captured iteration (cudaGraphGetNodes) */
    double fmax;            /* O8: max row norm of the NEB force of the last step (cell rows count as rows) */
    double barrier;         /* O8: E_{p*} - E_0 at the last evaluation */
    double dt, alpha;       /* FIRE state after the last step */
    double cell_factor;     /* lam actually used */
    double path_length;     /* sum_p |X_{p+1} - X_p| at the last evaluation */
} cfneb_status;

/* One row of the per-iteration record kept on the device (cfneb_get_history): what cfneb_get_status would have
 * reported had it been called right after that iteration. */
#define CFNEB_HISTORY_LEN 1024
typedef struct cfneb_history_entry {
    int64_t step;           /* status.steps after the iteration (1 = the first iteration of the band) */
    int64_t rebuilds;       /* neighbour-list rebuilds done so far */
    int32_t n_images;       /* P during the iteration */
    int32_t climb_index;    /* p* of the iteration, -1 if none */
    double fmax;            /* O8: max row norm of the NEB force of the iteration */
    double barrier;         /* O8: E_{p*} - E_0 at its evaluation */
    double dt, alpha;       /* FIRE state after it */
} cfneb_history_entry;

/* The scalar part of a checkpoint: the FIRE state of the band (O7; one state for the whole band, A3) and the
 * iteration counter.  first = 1: the next step skips the power test (A2). */
typedef struct cfneb_fire_state {
    double dt, alpha;
    int64_t steps;
    int32_t n_pos, first;
} cfneb_fire_state;

/* Kernel classes timed by cfneb_step_timed. */
enum {
    CFNEB_K_CELLPREP = 0,  /* K0  cell map D = sqrt(B), Cartesian positions */
    CFNEB_K_NEIGHBOR = 1,  /* K1  cell-list neighbour build (when it runs) */
    CFNEB_K_FORCE = 2,     /* K2  batched force / energy / virial (both passes for FS) */
    CFNEB_K_REDUCE = 3,    /* K4  ten segmented dot products per image */
    CFNEB_K_SCALAR = 4,    /* K5  tangent weights, climbing image, FIRE scalars, cell rows */
    CFNEB_K_UPDATE = 5,    /* K6  fused NEB force + cell-filter transform + FIRE update */
    CFNEB_NKERNELS = 6
};

/* Fill *prm with the defaults of O7 (FIRE: nmin 5, finc 1.1, fdec 0.5, astart 0.1, fa 0.99, dt0 0.1,
 * dtmax 1.0, maxstep 0.2), k_spring 1, climb 1, CELL_B, lam 1, skin 0.3, max_neighbors 160,
 * rebuild_every 0, LJ eps = sigma = 1, r_c = 2.5. */
CFNEB_API void cfneb_default_params(cfneb_params *prm);

/* Bytes of device workspace cfneb_create needs for n_atoms atoms and prm->max_images images
 * (0 on invalid arguments).  c4 (101306 atoms x 100 images, list capacity 224): 12.4 GB, of which 9.1 GB are the
 * neighbour lists. */
CFNEB_API size_t cfneb_workspace_bytes(int32_t n_atoms, const cfneb_params *prm);

/*
 * Create a band (two known endpoints; positions + lattice per image).
 *   pos_init/cell_init, pos_final/cell_final: HOST, N*3 and 9 doubles, Cartesian / rows = lattice vectors.
 *   n_images: P >= 3 including both endpoints, <= prm->max_images.
 *   path_or_null: HOST, optional explicit interior images, (P-2) blocks of (N*3 + 9) doubles
 *       (Cartesian positions then cell); if NULL the interior is linear in (R~, B) (or (R~, D) for CELL_D).
 *   dev_workspace: DEVICE pointer, 256-byte aligned, ws_bytes >= cfneb_workspace_bytes().
 *   cuda_stream: a cudaStream_t (may be NULL = legacy default stream; must not be capturing).
 * Maps inputs to generalized coordinates (O0) on the device, evaluates all P images once
 * (endpoint energies), builds neighbour lists and captures the step graph.  Synchronises.
 */
CFNEB_API int cfneb_create(cfneb_t **out, int32_t n_atoms, const double *pos_init, const double *cell_init,
                 const double *pos_final, const double *cell_final, int32_t n_images, const double *path_or_null,
                 const cfneb_params *prm, void *dev_workspace, size_t ws_bytes, void *cuda_stream);

/* Enqueue n_steps CFNEB iterations (K0-K6 of DESIGN.md; one force evaluation of every movable image
 * + one FIRE update each) as CUDA-graph launches on the stream.  Asynchronous: no host
 * synchronisation, no host<->device traffic. */
CFNEB_API int cfneb_step(cfneb_t *h, int32_t n_steps);

/*
 * n_steps iterations with the adaptive control step O9 (the rule of cfneb_adapt, reading A16) decided and
 * applied ON THE DEVICE after every adapt_every-th of them: segment lengths, at most one deletion and one midpoint
 * insertion, order-table edit and FIRE restart are kernels on the handle's stream, so a run with adaptive images
 * needs no host round trip either.  Asynchronous like cfneb_step; the host's view of P and of the order table is
 * refreshed by the next call that needs it (cfneb_get_status reports the device's P).  adapt_every >= 1.
 */
CFNEB_API int cfneb_step_adaptive(cfneb_t *h, int32_t n_steps, int32_t adapt_every, double d_insert, double d_delete);

/* Same iterations launched kernel by kernel with CUDA events between kernel classes; adds the
 * elapsed milliseconds per class, summed over the n_steps, to kernel_ms[CFNEB_NKERNELS] (HOST).
 * Synchronises.  For measurement only (bench.py roofline). */
CFNEB_API int cfneb_step_timed(cfneb_t *h, int32_t n_steps, double *kernel_ms);

/* Insert the midpoint of images (after_index, after_index+1) in generalized coordinates (O9);
 * resets the FIRE state (v = 0, dt = dt0).  The new image's energy is evaluated on the next step. */
CFNEB_API int cfneb_insert_image(cfneb_t *h, int32_t after_index);

/* Remove an interior image (not an endpoint, not the current climbing image); resets the FIRE state. */
CFNEB_API int cfneb_delete_image(cfneb_t *h, int32_t index);

/* Host-side control step of O9 (reading A16): at most one deletion (interior non-climbing image
 * minimising d_{q-1}+d_q, if below d_delete and P > 3) and one insertion (longest segment, if above
 * d_insert and P < max_images) with d_p = |X_{p+1} - X_p|.  Synchronises.  n_ins/n_del may be NULL. */
CFNEB_API int cfneb_adapt(cfneb_t *h, double d_insert, double d_delete, int32_t *n_ins, int32_t *n_del);

/*
 * Arc-length re-parametrisation of the band (the image distribution is "automatically adjusted ... based on
 * local spacing in configuration space"; reading A27): every interior image moves to arc length p L / (P - 1) along
 * the band's own polyline in the generalized coordinates X, s_p = sum_{q<p} |X_{q+1} - X_q|, by linear interpolation
 * on the segment that contains that point.  hold_climbing != 0: the climbing image of the last step stays where it is
 * and the images on each side of it are redistributed between it and their endpoint.  Endpoints never move; P and the
 * image order are unchanged; FIRE restarts (v = 0, dt = dt0) as after an insertion.  Runs as kernels on the handle's
 * stream: asynchronous, no host round trip, so it can sit between cfneb_step calls of a running band.  The moved
 * images' energies are NaN until the next step; their neighbour lists are kept while the move stays inside the skin.
 */
CFNEB_API int cfneb_reparametrize(cfneb_t *h, int32_t hold_climbing);

/* Segment lengths d_p = |X_{p+1} - X_p|, p = 0..P-2, at the current X (HOST, P-1 doubles). Synchronises. */
CFNEB_API int cfneb_get_segment_lengths(cfneb_t *h, double *d);

/*
 * Cell-filter FIRE relaxation of the two endpoints on the device (the step before the band in every
 * BASELINE.json config: "both endpoints cell-relaxed"; the paper's workflow starts from relaxed end states).
 * Each endpoint is relaxed as an independent structure in the band's generalized coordinates X = [R~ ; lam B] with
 * f = G (Eq. 12, 17; no tangent, no springs) and its own FIRE state (O7, step limit maxstep sqrt(N + 3)); an
 * endpoint stops when the max row norm of its G is below fmax_tol (tested before every update) and the call returns
 * when both have stopped or after max_steps updates.  The interior images are not touched while this runs.
 *   rebuild_band != 0: afterwards the band is rebuilt from the relaxed endpoints exactly as cfneb_create without an
 *       explicit path would: h0 := relaxed cell of image 0 (A7), lam (A13) recomputed, interior images linear in X,
 *       FIRE restarted, neighbour lists rebuilt, the iteration graph re-captured.
 *   rebuild_band == 0: only the endpoints change; FIRE of the band is restarted.
 * Outputs (each may be NULL): steps_done[2] updates taken per endpoint, fmax_out[2] and energy_out[2] at the final
 * states.  Synchronises.
 */
CFNEB_API int cfneb_relax_endpoints(cfneb_t *h, double fmax_tol, int32_t max_steps, int32_t rebuild_band,
                                    int32_t *steps_done, double *fmax_out, double *energy_out);

/* Current path: *n_images = P; pos P*N*3 Cartesian (R = R~ D), cells P*9 (h = h0 D, D = sqrt(B):
 * rotation-free), energies P (of the last evaluation; NaN for an image inserted since).
 * Any of pos/cells/energies may be NULL.  Synchronises. */
CFNEB_API int cfneb_get_path(cfneb_t *h, int32_t *n_images, double *pos, double *cells, double *energies);

/* Replace all P images from HOST Cartesian data (pos P*N*3, cells P*9; image 0's cell must equal h0).
 * This is a NEW PATH, not a resume: the FIRE state is reset (v = 0, dt = dt0, first step), and X is re-derived from
 * the Cartesian data (R~ = R D^-1, B = D D^T), so it need not equal bit for bit the X it was exported from -- to
 * continue a stopped band use cfneb_get_checkpoint / cfneb_set_state.  Endpoint energies are re-evaluated, interior
 * energies by the next cfneb_step / cfneb_get_forces (or on demand by cfneb_get_path).  Neighbour lists are kept: the
 * distance of the new coordinates from the stored ones is added to each image's displacement bound, so only images
 * that left their skin rebuild (editing a few images on the host rebuilds nothing else).  Synchronises. */
CFNEB_API int cfneb_set_path(cfneb_t *h, const double *pos, const double *cells);

/* Generalized coordinates X and FIRE velocities v, each P*(N+3)*3 (either may be NULL).  Read only. */
CFNEB_API int cfneb_get_state(cfneb_t *h, double *X, double *v);

/*
 * Checkpoint of the running band ("structural information is always kept and updated on GPU": this is the
 * way out and back in).  Everything the next iteration depends on, so that
 *     cfneb_get_checkpoint -> cfneb_destroy -> cfneb_create(same endpoints, same params, P images) -> cfneb_set_state
 * continues BIT FOR BIT as the uninterrupted band would have:
 *   X, v      P*(N+3)*3 each, as cfneb_get_state;
 *   X_list    P*(N+3)*3: the generalized coordinates at which each image's neighbour list was last built (the
 *             order of a list's entries fixes the summation order of the forces, so a resume replays the builds);
 *   list_aux  P*4: per image {max_i |R~_i - R~_i(build)|^2 at the last cell map, max_i |dR~_i|^2 of the last update,
 *             iterations since the build, pending} -- the staleness accounting that decides the next rebuild; pending
 *             is what calls made since the last iteration left for the next cell map: max_i |dR~_i|^2 of a
 *             cfneb_set_path / cfneb_set_state / cfneb_reparametrize move, or -1 for an image whose list must be
 *             rebuilt regardless (just inserted; its X_list row is then meaningless and cfneb_set_state ignores it).
 *             A checkpoint may therefore be taken at any point between two calls, not only after a plain step;
 *   fire      the FIRE scalars and the iteration counter.
 * All HOST, any may be NULL.  Read only; synchronises.
 */
CFNEB_API int cfneb_get_checkpoint(cfneb_t *h, double *X, double *v, double *X_list, double *list_aux,
                                   cfneb_fire_state *fire);

/*
 * Restore a checkpoint into a band of the same P, N and parameters.  X is copied as given (no round trip through
 * Cartesian coordinates), v as given (endpoint rows are ignored: zero); fire == NULL restarts FIRE (v is then zeroed).
 * With X_list and list_aux the neighbour lists are rebuilt at X_list and the accounting restored, which makes the
 * continuation bit-identical in a NEW handle (given its atom order: the same pos_init at cfneb_create).  With
 * X_list == NULL the handle's lists are kept and the distance of X from the stored coordinates is added to each image's
 * staleness bound (as cfneb_set_path does): handing a running band its own state back -- the host round trip of
 * bench.py's e2e loop -- rebuilds nothing and continues bit for bit; any other state continues to round-off
 * (summation order of the lists).
 * Endpoint energies are re-evaluated, interior energies by the next step (as cfneb_set_path).  Synchronises.
 * Errors: CFNEB_EINVAL (null X, X_list without list_aux, fire scalars out of range).
 */
CFNEB_API int cfneb_set_state(cfneb_t *h, const double *X, const double *v, const double *X_list,
                              const double *list_aux, const cfneb_fire_state *fire);

/*
 * One iteration of a band whose state is kept in HOST memory (pinned memory for full copy speed): X and v, each
 * P*(N+3)*3 as in cfneb_get_state, and the FIRE scalars go in, the iteration runs, and the new X, v and scalars come
 * back in the same buffers.  The same arithmetic, bit for bit, as
 *     cfneb_set_state(h, X, v, NULL, NULL, fire); cfneb_step(h, 1); cfneb_get_checkpoint(h, X, v, NULL, NULL, fire);
 * (the handle keeps its neighbour lists; see cfneb_set_state), but the upload is cut into n_blocks blocks of
 * consecutive images (0 = 10) sent on a second stream, and each block is evaluated -- cell map, list upkeep, forces:
 * an image needs only its own coordinates for that -- while the later blocks are still on their way; only the
 * reductions, the FIRE scalars and the update wait for the last block ("structural information is always kept and
 * updated on GPU", is the fast path; this is the way to step a band that does not live there).  Synchronises.
 * v == NULL: the velocities stay resident in the handle (an optimizer's internal state) and only the coordinates
 * travel, half the bytes; fire == NULL: the FIRE scalars stay resident as well.  Still the same arithmetic bit for bit
 * when X is the handle's own state handed back.
 * Errors: CFNEB_EINVAL (null h or X, scalars out of range), CFNEB_ERANGE (4096 images or more).
 */
CFNEB_API int cfneb_step_hosted(cfneb_t *h, double *X, double *v, cfneb_fire_state *fire, int32_t n_blocks);

/* Parity hook: evaluate forces at the CURRENT X without updating anything.  F: P*N*3 Cartesian forces
 * (Eq. 5), virial: P*9 (Eq. 8), f_neb: P*(N+3)*3 NEB force of Eq. 1 in generalized coordinates (zero rows
 * for endpoints), energies: P.  Any may be NULL.  Synchronises. */
CFNEB_API int cfneb_get_forces(cfneb_t *h, double *F, double *virial, double *f_neb, double *energies);

/* Parity hook: the ten K4 dot products of every image at the CURRENT X (Eq. 1; ref [13] via P:20), taken by
 * the band's own reduction (reduce_kernel + the second stage in scalar_kernel) in a dry evaluation that updates
 * nothing, and the generalized force they were taken with.  With tau+ = X_{p+1} - X_p, tau- = X_p - X_{p-1}:
 *   dots  P*10: {tau+.tau+, tau-.tau-, tau+.tau-, G.tau+, G.tau-, G.G, G.v, tau+.v, tau-.v, v.v} per image, all
 *               (N+3) x 3 components (cell rows included); endpoint rows are zero;
 *   coef  P*4:  {c1, c2, f.v, f.f} of K5's one-pass algebra, f = G + c1 tau+ + c2 tau- (zero for endpoints);
 *   G     P*(N+3)*3: generalized force [F D^T ; G_cell] (Eq. 12, 17) in the layout of cfneb_get_state (zero rows for
 *               endpoints).
 * Any may be NULL.  Synchronises. */
CFNEB_API int cfneb_get_dots(cfneb_t *h, double *dots, double *coef, double *G);

/*
 * The ten dot products of K4 for callers that cannot allocate device memory -- and cannot hand this library a
 * workspace to carve either: a plug-in inside a host MD / optimiser code that received its arrays and no allocator, a
 * process whose GPU memory was committed in full at start-up (a caching pool at its cap, a fixed MPS / MIG budget), a
 * latency-bound loop that may not take the device-wide synchronisation cudaMalloc implies.  The block partials of the
 * reduction live in a fixed array inside the library's own device image (640 KiB on every GPU that loads the library,
 * held until the process exits); the call itself performs no cudaMalloc, cudaFree or other allocating call.
 *   X, G, v: DEVICE pointers, n_images * n_dof doubles each, row-major [image][dof]: generalized coordinates,
 *       generalized forces and FIRE velocities of the band (the layouts of cfneb_get_state and of cfneb_get_dots' G
 *       with n_dof = 3 (N + 3); any n_dof >= 1 is accepted).  Read only; rows 0 and n_images-1 of G and v are not read.
 *   dots: DEVICE pointer, n_images * 10 doubles, written: per image the ten numbers listed at cfneb_get_dots, rows 0
 *       and n_images-1 zero.  Summation order is fixed: the same inputs give the same bits on every call.
 *   cuda_stream: the cudaStream_t to enqueue on (NULL = legacy default stream).  Asynchronous: returns once the two
 *       kernels are enqueued; `dots` is valid when the stream has reached that point.
 * Limits: 3 <= n_images <= CFNEB_NOALLOC_MAX_IMAGES (the size of the fixed scratch); a longer band is refused with
 * CFNEB_ERANGE and nothing is launched -- use a cfneb_create handle, whose scratch is sized by the caller's workspace.
 * The device that owns the pointers and the stream must be the CURRENT device of the calling thread.
 * First call on each device: the library looks up the device address of its scratch array (cudaGetSymbolAddress,
 * which may also make the runtime load the library's device code on that GPU).  That is one-time set-up, not part of
 * the steady state: make this first call before any CUDA stream capture is begun.
 * Sharing: one scratch array per GPU serves all calls.  A call rewrites every slot it later reads, so it needs no
 * clearing and is not affected by what the previous call left; but two calls that are in flight on the same GPU at the
 * same time (two streams, two host threads) write the same slots and corrupt each other.  Issue them on one stream
 * or order them with events.
 * Errors: CFNEB_EINVAL (NULL or non-device pointer, pointer of another device, n_images < 3, n_dof < 1), CFNEB_ERANGE
 * (n_images beyond the maximum), CFNEB_ECUDA; cfneb_band_dots_noalloc_error() returns the text of this thread's last
 * failure of this call ("" after a success).
 */
#define CFNEB_NOALLOC_MAX_IMAGES 128
CFNEB_API int cfneb_band_dots_noalloc(const double *X, const double *G, const double *v, int32_t n_images, int64_t n_dof,
                                      double *dots, void *cuda_stream);
CFNEB_API const char *cfneb_band_dots_noalloc_error(void);

/* Parity hook: neighbour list of one image as built on the device for the current X:
 * count[N], list[N*cap] (entry k of atom i at list[i*cap + k]), shift[N*cap*3]; r^ij = (s_j - s_i + n) h.
 * cap = prm->max_neighbors.  Forces a fresh build of that image.  Synchronises. */
CFNEB_API int cfneb_get_neighbors(cfneb_t *h, int32_t image, int32_t *count, int32_t *list, int32_t *shift);

/* Synchronise and report. */
CFNEB_API int cfneb_get_status(cfneb_t *h, cfneb_status *out);

/*
 * The convergence record of the last iterations (the paper's convergence and energy-barrier plots, P:144, P:152,
 * without a host synchronisation per step): K5 files one row per iteration in a ring of CFNEB_HISTORY_LEN rows in the
 * workspace, whoever launched the iteration (cfneb_step, cfneb_step_adaptive, cfneb_step_timed, cfneb_step_hosted), so
 * cfneb_step(h, 500) leaves 500 rows and this call is the only one that synchronises.
 *   out[i], i = 0..n-1: the iteration after which status.steps == first_step + i; bit for bit the fields of a
 *   cfneb_get_status taken at that point.  HOST, n entries.
 * Errors: CFNEB_ERANGE if first_step < 1, if first_step + n - 1 exceeds the iterations done, if a requested row has been
 * overwritten (more than CFNEB_HISTORY_LEN iterations ago) or was never written (the counter was moved by
 * cfneb_set_state); the sticky device error otherwise.  Synchronises.
 */
CFNEB_API int cfneb_get_history(cfneb_t *h, int64_t first_step, int32_t n, cfneb_history_entry *out);

CFNEB_API void cfneb_destroy(cfneb_t *h);
CFNEB_API const char *cfneb_strerror(int code);
CFNEB_API const char *cfneb_last_cuda_error(void);

/* Measurement utility: sustained fp64 FMA throughput of this GPU (TFLOP/s, 2 flops per DFMA) from a
 * register-resident DFMA chain kernel; the denominator of the force kernel's "alu" roofline. */
CFNEB_API int cfneb_util_fp64_peak(void *cuda_stream, double *tflops);

#ifdef __cplusplus
}
#endif
#endif /* CFNEB_H */

/* nnp.h -- C ABI of libnnp_b200: Behler-Parrinello neural-network-potential (NNP)
 * energy + force evaluation on one NVIDIA B200 (sm_100a).
 *
 * What it computes: the per-timestep NNP kernel of arXiv 2002.00054 section 3.1,
 * Fig. 1(b): step 1 atom-centred symmetry functions ("Gaussian
 * functions of neighbor distances with radial or angular character", L34), step 2
 * one small feed-forward network per atom giving the atomic energy, step 3 forces
 * from the gradient of the network w.r.t. the descriptors times the gradient of the
 * descriptors w.r.t. coordinates, with dG/dr recomputed instead of stored (L56-58,
 * L98, L124), preceded by a periodic cell-list neighbour build (L48, L116).
 * The paper prints no formulas; the exact definitions used (cosine cutoff, n2p2
 * type-2 radial and type-3 "narrow" angular functions, softplus networks) are listed
 * in DESIGN.md "Readings" and restated at nnp_sf below.
 *
 * Conventions
 *   - units: Angstrom, eV (whatever the weights encode); all floating point is FP64.
 *   - "device" pointers are CUDA device memory on the model's device; "host" pointers
 *     are ordinary (preferably pinned) host memory.
 *   - nothing here allocates per call except nnp_compute_host (library-owned, cached).
 *   - every function returns an nnp_status; no exceptions, no abort() across the ABI.
 *     Argument errors are returned synchronously.  Errors detected on the device
 *     (neighbour overflow, non-finite input) are reported by nnp_sync_status(), for every
 *     evaluation since the previous nnp_sync_status().
 *   - nnp_compute enqueues work on the caller's stream and returns without
 *     synchronising.  There is no CPU fallback: without a CUDA device every entry
 *     point that needs one returns NNP_ERR_CUDA.
 *   - a model is not thread-safe; use one model per host thread / stream.
 */
#ifndef NNP_H_
#define NNP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nnp_model nnp_model; /* opaque, owned by the library */

typedef enum {
    NNP_OK = 0,
    NNP_ERR_INVALID_ARG = 1,       /* null pointer, bad size, unsupported SF parameter */
    NNP_ERR_BOX_TOO_SMALL = 2,     /* some box length < 2*rc (minimum image would be ambiguous) */
    NNP_ERR_TYPE_RANGE = 3,        /* an atom type outside [0, n_elem)  (device-detected) */
    NNP_ERR_NEIGHBOR_OVERFLOW = 4, /* an atom has more neighbours than max_neighbors (device-detected) */
    NNP_ERR_WORKSPACE = 5,         /* workspace pointer null / misaligned / too small */
    NNP_ERR_CUDA = 6,              /* CUDA runtime error; see nnp_last_error */
    NNP_ERR_NONFINITE = 7,         /* NaN/Inf in positions (device-detected) */
    NNP_ERR_FORCE_RANGE = 9,       /* nnp_set_deterministic_forces: a force contribution beyond the fixed-point range
                                      (device-detected; forces of that call are incomplete) */
    NNP_ERR_LIMIT = 8              /* a well-formed request beyond a compile-time limit of this build: more than
                                      NNP_MAX_ELEMENTS elements, max_neighbors > NNP_MAX_NEIGHBORS, a hidden layer wider
                                      than NNP_MAX_HIDDEN_WIDTH, more than 8 weight layers, more than 128 radial / 512
                                      angular symmetry functions per element; nnp_last_error names the limit */
} nnp_status;

/* compile-time limits (NNP_ERR_LIMIT) */
#define NNP_MAX_ELEMENTS 4
#define NNP_MAX_NEIGHBORS 255
#define NNP_MAX_HIDDEN_WIDTH 256

/* One symmetry function of central element `central` (n2p2 numbering, C2-C5).
 *   kind 2 (radial):  G = sum_{j in N(i), t_j = e1} exp(-eta (r_ij - rs)^2) fc(r_ij)
 *   kind 3 (angular, narrow): with a=r_ij, b=r_ik, c=r_jk, cos = u.v/(ab),
 *       G = 2^(1-zeta) sum_{j<k in N(i), {t_j,t_k} = {e1,e2}, c < rc}
 *               (1 + lambda cos)^zeta  exp(-eta (a^2+b^2+c^2))  fc(a) fc(b) fc(c)
 *   kind 9 (angular, wide): the same without the r_jk terms,
 *       G = 2^(1-zeta) sum_{j<k in N(i), {t_j,t_k} = {e1,e2}} (1 + lambda cos)^zeta  exp(-eta (a^2+b^2))  fc(a) fc(b)
 *       (every pair of neighbours is a triplet; such functions run as passes of their own, NNP_KERNELS_MULTI)
 *   fc(r) = (cos(pi r / rc) + 1)/2 for r < rc, else 0;  N(i) = { j != i : r_ij^2 < rc^2 }.
 * Constraints (else NNP_ERR_INVALID_ARG): eta >= 0; kinds 3 and 9 need lambda = +1 or -1 and
 * zeta an integer in [1, 64]; rs is used by kind 2 only.  The order of the entries with
 * equal `central` is the order of that element's descriptor vector G (= network input). */
typedef struct {
    int32_t central;
    int32_t kind;
    int32_t e1, e2;
    double eta, rs, lambda, zeta;
} nnp_sf;

/* Create a model on CUDA device `cuda_device` ("potential parameters, masses, symmetry-function
 * parameters, NN weights and biases" are per-type tables; L58: n2p2-based initialisation is replaced by these arguments).
 *   n_elem        number of elements (1..NNP_MAX_ELEMENTS, more: NNP_ERR_LIMIT); atom types are indices into elem_names.
 *   elem_names    [n_elem] NUL-terminated names (copied; informational).
 *   rc            cutoff radius (> 0), one for all symmetry functions.
 *   sf            [n_sf] symmetry functions, all elements together (copied).
 *   n_layers      [n_elem] number of weight layers of each element's network (>= 1).
 *   layer_sizes   [n_elem] -> [n_layers[e]+1] sizes; first = number of SFs with central == e,
 *                 last = 1.  Hidden widths <= 256.
 *   weights       [n_elem] -> flat row-major  W1[out][in], b1[out], W2, b2, ...  (copied).
 *                 Hidden layers use softplus log(1+e^x); the output layer is linear.
 * All inputs are host memory and are not referenced after return. */
nnp_status nnp_create(nnp_model** out, int32_t n_elem, const char* const* elem_names, double rc,
                      int32_t n_sf, const nnp_sf* sf, const int32_t* n_layers,
                      const int32_t* const* layer_sizes, const double* const* weights,
                      int32_t cuda_device);

/* Which kernels a symmetry-function table would run on (host only, no CUDA call; nnp_create takes the same
 * decision): kernels_out[c] for every central element c --
 *   NNP_KERNELS_BASE12 / NNP_KERNELS_WIDE32  the lane-owned kernels specialised for BASELINE.json's two angular tables,
 *   NNP_KERNELS_FREE32 / NNP_KERNELS_FREE16  the lane-owned kernels for any table with <= 4 (FREE16: <= 2) distinct
 *                        angular eta values, lambda = +-1, zeta in one exponent menu {z0, 2 z0, 4 z0, zx} (any integers, e.g.
 *                        {1, 2, 4, 16}, {1, 4}, {1, 2, 4, 3}), narrow (kind 3) functions only, no (eta, lambda, zeta) twice per
 *                        pair group,
 *   NNP_KERNELS_MULTI    the same lane-owned free-eta kernels in several passes: any number of eta values (four per pass),
 *                        wide functions (kind 9; passes of their own), any integer zeta (one pass per exponent menu) and,
 *                        after nnp_set_sf_cutoffs, angular functions of several cutoff radii (one radius per pass), at most
 *                        8 passes; otherwise the conditions of FREE32,
 *   NNP_KERNELS_GENERIC  everything else (more passes, a function listed twice, eta * 3 rc^2 > 700, no angular functions).
 * Returns NNP_ERR_INVALID_ARG for a table nnp_create would reject (message: nnp_last_error(NULL)). */
#define NNP_KERNELS_GENERIC 0
#define NNP_KERNELS_BASE12 1
#define NNP_KERNELS_WIDE32 2
#define NNP_KERNELS_FREE32 3
#define NNP_KERNELS_FREE16 4
#define NNP_KERNELS_MULTI 5
nnp_status nnp_table_kernels(int32_t n_elem, double rc, int32_t n_sf, const nnp_sf* sf, int32_t* kernels_out);

/* Free the model and everything the library allocated for it.  NULL is allowed. */
void nnp_destroy(nnp_model* m);

/* Upper bound on neighbours per atom the kernels provision for (PAPER.md L48 / L116: the per-atom neighbour list;
 * default 160 -- the water-like workloads average 91, Poisson tail < 150 at 2.1 M atoms).  Range 16..NNP_MAX_NEIGHBORS
 * (below 16: NNP_ERR_INVALID_ARG; above 255: NNP_ERR_LIMIT -- the kernels address neighbour slots with 8 bits).  The value
 * also selects kernels: up to 32 the small-neighbourhood kernels (eight lanes per centre; up to 24 with smaller per-centre
 * shared memory -- the paper's Ni system has 18 neighbours, PAPER.md L70 / L96), up to 64 one warp per centre, else two. */
nnp_status nnp_set_max_neighbors(nnp_model* m, int32_t max_neighbors);

/* Neighbour-list reuse with a Verlet skin ("neighbor list", L116; an MD code rebuilds its
 * list only every few steps).  skin in Angstrom, 0 <= skin <= rc; 0 (the default) = every nnp_compute bins, sorts and
 * searches the cells again.  With skin > 0 nnp_compute keeps, in the CALLER'S workspace, the sorted order and a
 * candidate list of radius rc + skin from the last rebuild, and every call
 *   1. checks on the device whether any atom has moved more than skin/2 since that rebuild (minimum image) or changed
 *      its type -- then, or when the workspace pointer, n_atoms or the box differ from the last call (host-side check),
 *      it rebuilds: sort + cell search with rc + skin;
 *   2. filters the exact list N(i) = { j : r_ij < rc } of THIS call's positions out of the candidate list with the same
 *      FP64 predicate as a fresh build.
 * Results are those of skin = 0: the same neighbour sets bit for bit, energies and forces up to summation order.
 * The decision is taken on the device, so the launch sequence is fixed (nnp_md_run replays it as a CUDA graph).
 * The caller must leave the workspace content untouched between calls (or call nnp_invalidate_neighbors);
 * nnp_workspace_bytes grows by the candidate list (about max_neighbors * ((rc+skin)/rc)^3 * 4 B per atom) -- query it
 * AFTER this call.  Box lengths must be >= 2 (rc + skin).  A candidate row that overflows reports
 * NNP_ERR_NEIGHBOR_OVERFLOW like an exact row.  Errors: NNP_ERR_INVALID_ARG (skin < 0, not finite, > rc). */
nnp_status nnp_set_neighbor_skin(nnp_model* m, double skin);
/* Forget the candidate list: the next nnp_compute rebuilds (use after writing into the workspace). */
nnp_status nnp_invalidate_neighbors(nnp_model* m);
/* Calls and rebuilds since nnp_set_neighbor_skin (synchronises the stream of the last call; host pointers). */
nnp_status nnp_get_neighbor_rebuilds(nnp_model* m, int64_t* n_calls, int64_t* n_rebuilds);

/* Bytes of device workspace nnp_compute needs for n_atoms (0 on error): sorted coordinates, neighbour rows, G and
 * dE/dG rows, screening masks -- about 2.9 KB per atom for the base-52 model.  The derivative tensor dG/dr is never
 * stored ("store and move as little data as possible, recomputing where necessary"; L82: what lets
 * 2 M atoms fit one GPU), so this is the whole memory footprint of an evaluation. */
size_t nnp_workspace_bytes(const nnp_model* m, int64_t n_atoms);

/* One energy + force evaluation (Fig. 1(b) steps 1-3 after the neighbour build).
 *   d_pos        [n_atoms][3] device, any real coordinates (wrapped into the box internally)
 *   d_type       [n_atoms]    device, element index per atom
 *   box          [3] HOST, orthorhombic box lengths, origin 0; each must be >= 2*rc
 *   d_e_atom     [n_atoms]    device out, atomic energies E_i, caller's atom order
 *   d_e_total    [1]          device out, E = sum_i E_i (deterministic summation order)
 *   d_force      [n_atoms][3] device out, F_m = - sum_i sum_s dE_i/dG_is * dG_is/dr_m
 *   d_workspace  device, 256-byte aligned, >= nnp_workspace_bytes(m, n_atoms); owned by the
 *                caller; it also holds the neighbour list / G read by the nnp_get_* calls, so
 *                keep it alive until those are done.
 *   cuda_stream  a cudaStream_t (NULL = default stream); all work is enqueued there.
 * n_atoms == 0 is allowed (writes e_total = 0). */
nnp_status nnp_compute(nnp_model* m, int64_t n_atoms, const double* d_pos, const int32_t* d_type,
                       const double box[3], double* d_e_atom, double* d_e_total, double* d_force,
                       void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/* Same evaluation with HOST buffers: copies pos/type to the device, runs nnp_compute on an
 * internal stream with library-owned (cached) device buffers, copies e_atom / e_total / force
 * back and synchronises.  Returns device-detected errors too. */
nnp_status nnp_compute_host(nnp_model* m, int64_t n_atoms, const double* h_pos, const int32_t* h_type,
                            const double box[3], double* h_e_atom, double* h_e_total, double* h_force);

/* ---- model generality (n2p2 models scale / centre their symmetry functions and may use
 * tanh).  Both settings apply to the following nnp_compute calls; defaults: no scaling, softplus.
 * nnp_set_sf_scaling: the network of element `elem` reads x_s = h_scale[s] * (G_s - h_shift[s]) instead of G_s
 *   (HOST arrays of the element's symmetry-function count, in G order; both NULL = back to identity).
 *   nnp_get_sf still returns the unscaled G, nnp_get_dedg returns dE/dG (= scale * dE/dx).  Synchronises the device.
 * nnp_set_activation: hidden-layer activation of every element; the output layer stays linear.
 * nnp_set_sf_cutoffs: per-SF cutoff radii (n2p2 gives every symmetry function its own rc): h_rc is a HOST array
 *   of n_sf radii in the order of the `sf` table of nnp_create, each 0 < h_rc[s] <= rc (else NNP_ERR_INVALID_ARG);
 *   SF s then uses fc(r; h_rc[s]) = (cos(pi r / h_rc[s]) + 1)/2 for r < h_rc[s], else 0 -- for r_ij, r_ik and, in
 *   kind 3, for r_jk (which must be < h_rc[s]) -- on the neighbourhood of the global rc.  NULL = back to the one
 *   global rc.  An element whose ANGULAR functions have radii other than rc runs on the multi-pass kernels
 *   (NNP_KERNELS_MULTI) if its table fits them, else on the generic kernels; radii on radial functions alone leave the
 *   choice of kernels as it was.
 *   Synchronises the device. */
#define NNP_ACT_SOFTPLUS 0
#define NNP_ACT_TANH 1
nnp_status nnp_set_sf_scaling(nnp_model* m, int32_t elem, const double* h_shift, const double* h_scale);
nnp_status nnp_set_activation(nnp_model* m, int32_t kind);
nnp_status nnp_set_sf_cutoffs(nnp_model* m, int32_t n_sf, const double* h_rc);

/* ---- mixed precision (the paper does not state its precision).  OPT-IN, never the default:
 * NNP_PRECISION_MIXED stages the neighbourhood of a centre in FP32 and evaluates the angular symmetry functions and
 * their force terms per triplet in FP32 (hardware exponential, degree-5 cutoff polynomials); the neighbour list and
 * its predicate, the minimum-image geometry, the radial symmetry functions, the networks, the reduction of the
 * symmetry-function sums over the lanes and every global force / energy accumulation stay FP64.  It applies to elements
 * whose table has one of BASELINE.json's two angular shapes (NNP_KERNELS_BASE12 / NNP_KERNELS_WIDE32) with
 * eta_0 rc^2 <= 0.05 and 64 < max_neighbors (centres with more than 160 neighbours stay FP64); every other element
 * silently keeps FP64.  The results no longer meet
 * BASELINE.json's tolerances (measured on the water-like configs: DESIGN.md section 6c); energies stay bit-reproducible. */
#define NNP_PRECISION_F64 0
#define NNP_PRECISION_MIXED 1
nnp_status nnp_set_precision(nnp_model* m, int32_t mode);

/* ---- bit-reproducible forces (BASELINE.json north_star: forces are accumulated "either atomic-free via per-atom gather or
 * with warp-aggregated atomics"; "thread-safe atomics as needed for ... force updates").  By default every centre
 * adds its contributions to the neighbours' forces with FP64 atomics: the ~180 additions per atom happen in an order that
 * differs from run to run, so forces repeat only to ~1e-13 eV/A (energies are always bit-reproducible).  With
 * nnp_set_deterministic_forces(m, 1) every contribution is rounded to a multiple of 2^-40 eV/A (9.1e-13) and accumulated as a
 * 64-bit integer; integer addition is associative, so the forces are the same bits on every run, at the same speed.  A
 * contribution beyond +-2^22 eV/A (coincident atoms) is reported as NNP_ERR_FORCE_RANGE by nnp_sync_status. */
nnp_status nnp_set_deterministic_forces(nnp_model* m, int32_t enabled);

/* ---- MD loop around the path (the implementation is checked by energy
 * conservation in an NVE run).  Velocity Verlet, everything on the device:
 *     v += (dt/2) F/m ;  x += dt v ;  F = nnp_compute(x) ;  v += (dt/2) F/m
 * Units: A, eV, amu, fs  (1 eV/(A amu) = NNP_ACC_UNIT A/fs^2).
 *
 * nnp_md_run advances n_steps steps.  On entry d_force must hold the forces of d_pos (call nnp_compute
 * first); on return d_pos / d_vel / d_force / d_e_atom / d_e_total belong to the last step.  Positions are
 * NOT wrapped (nnp_compute wraps internally).  The neighbour list is rebuilt every step, or -- after
 * nnp_set_neighbor_skin -- when an atom has moved half the skin (decided on the device, also inside the graph replay).
 *   h_mass   [n_elem] HOST, masses in amu, by element index
 *   d_vel    [n_atoms][3] device, in/out, A/fs
 * Everything is enqueued on cuda_stream; no synchronisation inside (except once at the start if the graph of a
 * previous run is still alive).  With n_steps >= 4, a non-NULL stream and per-stage timing off, steps 2..n are
 * replayed from a CUDA graph of one step captured on that stream (small systems are launch-latency bound).
 * nnp_md_kinetic_energy: *d_ekin (device, [1]) = sum_i m_i |v_i|^2 / (2 NNP_ACC_UNIT) in eV, deterministic
 * summation order; d_workspace as for nnp_compute (only its energy-partials scratch is touched, the exports of
 * the last nnp_compute stay valid). */
#define NNP_ACC_UNIT 9.648533215665327e-3 /* (1.602176634e-19 J/eV) / (1.66053906660e-27 kg/amu) * 1e-10, CODATA 2018 */
nnp_status nnp_md_run(nnp_model* m, int32_t n_steps, double dt_fs, const double* h_mass, int64_t n_atoms,
                      double* d_pos, double* d_vel, const int32_t* d_type, const double box[3],
                      double* d_e_atom, double* d_e_total, double* d_force,
                      void* d_workspace, size_t workspace_bytes, void* cuda_stream);
nnp_status nnp_md_kinetic_energy(nnp_model* m, const double* h_mass, int64_t n_atoms, const double* d_vel,
                                 const int32_t* d_type, double* d_ekin, void* d_workspace, size_t workspace_bytes,
                                 void* cuda_stream);

/* nnp_md_kinetic_energy for callers that cannot allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): the same quantity (the energy-conservation check of an NVE
 * run; same arithmetic and summation order, same bits) WITHOUT a workspace.  The block sums live in a static device
 * array inside the library: 128 KB that every GPU which loads the library holds until the process exits.  The call
 * makes no cudaMalloc / cudaFree and calls no allocating library routine; it enqueues two kernels on cuda_stream and
 * does not synchronise.
 *   h_mass [n_elem] HOST (amu);  d_vel [n_atoms][3], d_type [n_atoms], d_ekin [1] DEVICE, caller-owned.
 *   n_atoms <= NNP_NOALLOC_MAX_ATOMS, beyond: NNP_ERR_LIMIT and nothing is launched.
 * Every call on a device shares the array (a call overwrites what it reads; nothing needs clearing between calls):
 * calls that OVERLAP on the GPU -- different streams without an ordering between them, also from different models --
 * race on it.  Errors: NNP_ERR_INVALID_ARG (null pointers, n_atoms < 0, bad masses), NNP_ERR_LIMIT, NNP_ERR_CUDA. */
#define NNP_NOALLOC_MAX_ATOMS 4194304
nnp_status nnp_md_kinetic_energy_noalloc(nnp_model* m, const double* h_mass, int64_t n_atoms, const double* d_vel,
                                         const int32_t* d_type, double* d_ekin, void* cuda_stream);

/* Synchronise the stream of the last nnp_compute / nnp_md_run and return the device-side status of EVERY
 * evaluation enqueued since the previous nnp_sync_status (a sticky device word owned by the model: a neighbour
 * overflow or a non-finite position in step 3 of a 100-step nnp_md_run, or in the first of several nnp_compute
 * calls enqueued back to back, is still reported).  Reading clears the word.  Precedence when several flags are
 * set: NNP_ERR_NONFINITE, NNP_ERR_TYPE_RANGE, NNP_ERR_NEIGHBOR_OVERFLOW, NNP_ERR_FORCE_RANGE. */
nnp_status nnp_sync_status(nnp_model* m);

/* Debug / parity exports of the LAST nnp_compute (they synchronise its stream first): the neighbour list of
 * PAPER.md L48 / L116 ("random access (neighbor list)"), the descriptors of step 1 and the network gradient
 * dE/dG of steps 2-3 (L40, Fig. 1(b)).  Atom indices and row order are the CALLER's; all pointers are device memory.
 *   nnp_get_neighbor_counts: d_counts[n_atoms] = |N(i)|.
 *   nnp_get_neighbors: d_offsets[n_atoms+1] (exclusive prefix sum of the counts) and
 *                      d_idx[total] with every row sorted ascending.  d_idx may be NULL to get
 *                      offsets only; `idx_capacity` = number of int32 entries d_idx can hold.
 *   nnp_get_sf / nnp_get_dedg: [n_atoms][g_stride] with g_stride = nnp_g_stride(m)
 *                      (= max SFs per element; unused tail entries are 0). */
nnp_status nnp_get_neighbor_counts(nnp_model* m, int32_t* d_counts);
nnp_status nnp_get_neighbors(nnp_model* m, int64_t* d_offsets, int32_t* d_idx, int64_t idx_capacity);
nnp_status nnp_get_sf(nnp_model* m, double* d_G);
nnp_status nnp_get_dedg(nnp_model* m, double* d_dEdG);
int32_t nnp_g_stride(const nnp_model* m);

/* Per-stage device times of nnp_compute: the time split the paper reports per step (Fig. 5:
 * symmetry functions / network / force; force "up to 60 %", network "a minor part").  Off by default (no events recorded).
 * ms[NNP_N_STAGES]: 0 wrap+bin+sort, 1 neighbour list, 2 symmetry functions,
 * 3 networks fwd+bwd, 4 forces, 5 reduce+un-permute.  Synchronises the stream. */
#define NNP_N_STAGES 6
nnp_status nnp_set_timing(nnp_model* m, int32_t enabled);
nnp_status nnp_get_timings(nnp_model* m, double* ms);

/* Number of kernels the last nnp_compute / nnp_md_run launched (launch accounting of the benchmark; every
 * PAPER.md L98 "parallel_for" of the reference is a launch here too). */
int32_t nnp_last_launch_count(const nnp_model* m);

/* 1 if the model's angular symmetry functions run on a specialised kernel, 0 if on the
 * generic (slower, any-table) kernel. */
int32_t nnp_uses_fast_path(const nnp_model* m);

/* Measure the FP64 FMA issue rate of the device (independent DFMA chains on every SM; the path is bound by the
 * FP64 ALUs, so this is the measured roofline denominator next to the derived one):
 * thread-level DFMA instructions per second, *dfma_per_s = best 10-launch burst,
 * *dfma_per_s_sustained (may be NULL) = mean over the whole `seconds`.  Roofline denominator. */
nnp_status nnp_measure_fp64_peak(int32_t cuda_device, double seconds, double* dfma_per_s,
                                 double* dfma_per_s_sustained);

/* Last error text for this model (never NULL).  nnp_create failures: pass NULL. */
const char* nnp_last_error(const nnp_model* m);

/* "major.minor" of this library. */
const char* nnp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* NNP_H_ */

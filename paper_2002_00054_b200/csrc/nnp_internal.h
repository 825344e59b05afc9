// nnp_internal.h -- structures shared by the CUDA translation units of libnnp_b200.
// Not part of the public ABI (that is include/nnp.h).  Shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>

#include "nnp.h"

namespace nnp {

constexpr int MAX_ELEM = 4;
constexpr int MAX_PAIR = MAX_ELEM * (MAX_ELEM + 1) / 2;   // unordered neighbour-element pairs
constexpr int MAX_ETA = 4;        // distinct angular etas on the specialised path
constexpr int MAX_RAD_TOTAL = 128;  // radial SFs per central element (all neighbour elements)
constexpr int MAX_ANG_TOTAL = 512;  // angular SFs per central element (all pairs)
constexpr int MAX_LAYERS = 8;
constexpr int MAX_WIDTH = 256;

// Device-detected status bits (Workspace::status[0] is an OR of these)
enum : int { ST_TYPE_RANGE = 1, ST_NBR_OVERFLOW = 2, ST_NONFINITE = 4, ST_FORCE_RANGE = 8 };

// index of the unordered element pair (a <= b) among E elements
__host__ __device__ inline int pair_index(int a, int b, int n_elem) {
    return a * n_elem - (a * (a - 1)) / 2 + (b - a);
}

struct RadialSF {
    double eta, rs;
    int32_t g;       // position in the element's G vector
    int32_t pad;
    double rc2, k2;  // this SF's cutoff: rc_s^2 and (pi / (2 rc_s))^2 (read only when ElemProgram::per_sf_rc)
};

struct AngularSF {
    double eta;
    double coef;     // 2^(1-zeta)
    int32_t g;
    int32_t izeta;   // integer zeta
    int32_t lam;     // +1 / -1
    int32_t wide;    // 1: wide angular SF (n2p2 kind 9: no r_jk term, no r_jk cutoff); generic kernels only
    double rc2, k2;  // this SF's cutoff: rc_s^2 and (pi / (2 rc_s))^2 (read only when ElemProgram::per_sf_rc)
};

// Angular kernel variants.  Specialised variants bake the (eta ratio, lambda, zeta) structure
// of a pair group into the kernel; ANG_GENERIC walks the AngularSF list (any table).
enum AngVariant : int { ANG_GENERIC = 0, ANG_BASE12 = 1, ANG_WIDE32 = 2, ANG_FREE32 = 3, ANG_FREE16 = 4, ANG_MULTI = 5, ANG_NVARIANT = 6 };

// One sweep of the free-eta lane-owned kernels (SpecFree16 / SpecFree32) over the triplets of a centre: up to four
// eta values that share ONE cutoff radius.  A table with more eta values, or with angular symmetry functions of
// several radii (n2p2 gives every symmetry function its own rc), with wide functions or with zeta values outside
// {zeta0, 2 zeta0, 4 zeta0, zeta_x} for one pair (zeta0, zeta_x), runs as several passes -- G entries are independent and the forces are additive
// over the symmetry functions.  ANG_FREE16 / ANG_FREE32 = one pass at the
// global rc; ANG_MULTI = anything else that fits MAX_PASS passes.
// hand-over of the pair lists in k_small.cu: per centre [0] = 0 if valid, [1 + pair group] = entries of the group, [16 ..) the entries
constexpr int SMALL_LIST_U16 = 256;
constexpr int SMALL_LIST_HDR = 16;
constexpr int MAX_PASS = 8;
struct AngPass {
    double eta[MAX_ETA];
    double rc2, k2;                  // the pass's cutoff: rc_p^2, (pi / (2 rc_p))^2
    int32_t n_eta;
    int32_t spec;                    // ANG_FREE16 (<= 2 eta values) or ANG_FREE32
    int32_t own_rc;                  // 1: rc_p differs from the global rc (slots beyond rc_p are switched off while staging)
    int32_t wide;                    // 1: a pass of WIDE angular functions (n2p2 kind 9): no r_jk term, no r_jk cutoff -- every pair
                                     // of neighbours of the two elements is a triplet (no screening)
    int32_t zeta0;                   // menu bits 0, 1, 2 of this pass stand for zeta = zeta0, 2 zeta0, 4 zeta0: the kernels raise
                                     // (1 +- cos) to zeta0 first (a warp-uniform square-and-multiply loop) and square from there
    int32_t zeta_x;                  // menu bit 4 stands for zeta = zeta_x: 16 zeta0 (two more squarings) or any other exponent
                                     // (raised on its own by square-and-multiply)
    int32_t n_ang[MAX_PAIR];         // symmetry functions of pair group p in this pass (0: the group is skipped)
    int16_t g[MAX_PAIR][MAX_ETA][16];   // G index of menu entry (eta slot, bit); -1 = absent
};
// host-side summary for the launchers
struct PassInfo {
    int n_pass[MAX_ELEM];
    int spec[MAX_ELEM][MAX_PASS];
    int radial_own[MAX_ELEM];        // the element's radial functions carry their own cutoff radii (ElemProgram::per_sf_rc)
    int fixed_forces;                // nnp_set_deterministic_forces: fixed-point global force accumulation (force_add)
};

// Symmetry-function program of ONE central element; lives in device memory (model-owned).
struct ElemProgram {
    int32_t n_sf;
    int32_t n_elem;
    int32_t variant;                 // AngVariant
    int32_t tiny_exp;                // specialised path: eta_0 rc^2 <= 0.05 -> exp_tiny() for exp(-eta_0 r^2)
    int32_t per_sf_rc;               // 1: some SF of this element has its own cutoff radius (nnp_set_sf_cutoffs); generic kernels
    int32_t n_eta;                   // (unused since the passes; kept for layout)
    int32_t n_pass;                  // free-eta kernels: passes in use (pass[0 .. n_pass))
    int32_t n_rad[MAX_ELEM];         // radial SFs for neighbour element e
    int32_t rad_off[MAX_ELEM];       // first index into rad[]
    int32_t n_ang[MAX_PAIR];         // angular SFs of pair group p
    int32_t ang_off[MAX_PAIR];       // first index into ang[]
    // specialised path: eta values (shared by all groups of the element) and, per group,
    // the G index of menu entry (eta slot e, bit b): bits 0..6 lambda=+1 zeta=2^b, 8..14 lambda=-1
    double ang_eta[MAX_ETA];
    int16_t ang_g[MAX_PAIR][MAX_ETA][16];
    RadialSF rad[MAX_RAD_TOTAL];
    AngularSF ang[MAX_ANG_TOTAL];
    AngPass pass[MAX_PASS];
};

// Small networks (two hidden layers of width <= 32, <= 80 inputs) also travel in the KERNEL PARAMETER block
// (k_mlp_reg, k_mlp.cu): warp-uniform weights then come through the constant cache into uniform registers
// instead of through the load/store pipe.  Hidden widths are padded to 32 with zero weights.
constexpr int MLP_REG_H = 32;
constexpr int MLP_REG_MAXW = 3700;
struct MlpRegWeights {
    int32_t n_in, n1, n2, pad;
    double w[MLP_REG_MAXW];          // W1[n_in][32] | b1[32] | W2[32][32] (input-major) | b2[32] | w3[32] | b3
};

// One element's network in device memory.  `weights` holds, per layer l (all blocks padded to
// multiples of 4 doubles, zero filled): WT_l [n_in][round4(n_out)] (transposed, forward pass),
// W_l [n_out][round4(n_in)] (backward pass), b_l [round4(n_out)].
struct NetDesc {
    int32_t n_layers;                // weight layers
    int32_t sizes[MAX_LAYERS + 1];
    int32_t wt_off[MAX_LAYERS];
    int32_t w_off[MAX_LAYERS];
    int32_t b_off[MAX_LAYERS];
    const double* weights;           // device
    // model generality: network input x_s = sf_scale[s] * (G_s - sf_shift[s]); device arrays
    // [sizes[0]] or nullptr (identity); activation 0 = softplus, 1 = tanh (hidden layers; output linear)
    const double* sf_shift;
    const double* sf_scale;
    int32_t activation;
    const MlpRegWeights* reg;        // HOST memory (model-owned) or nullptr: parameter-block copy for k_mlp_reg
};

// Cell grid of one nnp_compute call (host-built, passed by value).
// Cells are at least rc / hw wide and the neighbour search visits the (2 hw + 1)^3 stencil: hw = 2 cuts the candidates
// per atom from 27 rc^3 rho to 15.6 rc^3 rho (583 -> 337 for the water-like systems); make_grid takes hw = 1 when such
// cells would hold fewer than 1.5 atoms (the search runs one warp per cell and amortises its bookkeeping over the cell's atoms).
struct Grid {
    double box[3], half[3], inv_cs[3];
    int32_t nc[3];
    int32_t ncell;
    int32_t hw;                      // stencil half-width: cells are >= rc / hw wide
    int32_t span[3];                 // hw if nc >= 2 hw + 1, else 0 (the stencil is all nc cells)
};

struct Workspace {
    double *sx, *sy, *sz;            // [N] wrapped coordinates, sorted by (element, cell, original index)
    double *tx, *ty, *tz;            // [N] staging for the sort
    int32_t *perm, *tperm;           // [N] sorted position -> original index
    int32_t *key, *rank, *tkey;      // [N]
    int32_t *cell_start;             // [n_elem * ncell + 1]
    int32_t *scan_tmp;               // block sums of the scans
    int32_t *nbr;                    // [N][stride] neighbour positions (sorted space), grouped by element
    int32_t *nbr_cnt;                // [N][MAX_ELEM] neighbours of each element
    // neighbour-skin mode (nnp_set_neighbor_skin; absent from the layout otherwise).  These, perm and cell_start are the
    // state a call that does not rebuild relies on: the caller keeps the workspace intact between calls.
    int32_t *snbr;                   // [N][sstride] candidate list of the last rebuild (radius rc + skin), grouped by element
    int32_t *snbr_cnt;               // [N][MAX_ELEM]
    double *bx, *by, *bz;            // [N] wrapped positions at the last rebuild, sorted order
    int32_t *skin_flag;              // device word: this call rebuilds (set by the host or by k_skin_check)
    int32_t *skin_stats;             // model-owned: [0] calls, [1] rebuilds since nnp_set_neighbor_skin
    uint16_t *slist;                 // small-neighbourhood kernels only (row stride <= 32, else null): [N][SMALL_LIST_U16] the compacted
                                     // (j, k) lists of a centre, handed from k_sf_small to k_force_small (k_small.cu)
    double *G, *dEdG;                // [N][g_stride], sorted order
    double *e_sorted;                // [N]
    double *f_sorted;                // [N][3]
    // masks handed from the symmetry-function kernel to the force kernel (fast paths): the SF kernel
    // screens the (j,k) candidates of every centre anyway; it stores the mask words of centre i in the
    // force kernel's (j-major) order at gmask[word_off[i] ..), if they fit the budget
    int32_t *big_list;               // [N] sorted positions of the centres with more than 128 neighbours (count: status[2])
    int32_t *nw;                     // [N] mask words of centre i
    int64_t *word_off;               // [N+1] exclusive prefix of nw
    int64_t *word_tmp;               // scan scratch
    uint32_t *gmask;                 // [gmask_cap]
    int64_t gmask_cap;
    double *partial;                 // [n_partial] block sums of the energy
    int32_t *status;                 // [4]; word 0 = flags of this nnp_compute, word 2 = length of big_list (all cleared by launch_sort)
    int32_t *sticky;                 // model-owned word: flags of every call since the last nnp_sync_status (set by nnp_compute, not by ws_layout)
    int64_t n_keys_cap;
    int64_t scan_tmp_len;
    int64_t n_partial;
    size_t bytes;
};

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-DEVICE attribute: opt a kernel instantiation in once per
// device it is launched on (`done` = one static bit mask per instantiation, indexed by the current device).  A
// failure stays in the runtime's last-error slot and is returned by the cudaGetLastError() at the end of nnp_compute.
template <class K>
inline void opt_in_smem(K kernel, unsigned long long* done, int bytes = 200 * 1024) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return;
    if (dev >= 0 && dev < 64 && ((*done >> dev) & 1ull)) return;
    if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) == cudaSuccess && dev >= 0 && dev < 64)
        *done |= 1ull << dev;
}

// Global force accumulation of the force kernels (their parameter blocks carry f_sorted, fixed, status, sticky).
// Default: FP64 atomics (RED.ADD.F64) -- the order of the ~180 additions per atom is not fixed, the forces repeat to ~1e-13.
// fixed = 1 (nnp_set_deterministic_forces): every contribution is rounded to a multiple of 2^-40 eV/A (9.1e-13) and added
// as a 64-bit INTEGER -- integer addition is associative, so the sums are bit-reproducible whatever the order; range
// +-2^22 eV/A per contribution (beyond: ST_FORCE_RANGE), +-2^23 per sum.  launch_finalize converts back.
constexpr double FORCE_FIXED_SCALE = 1099511627776.0;             // 2^40
constexpr double FORCE_FIXED_INV = 1.0 / 1099511627776.0;
constexpr double FORCE_FIXED_LIMIT = 4194304.0;                   // 2^22
#ifdef __CUDACC__
__device__ __forceinline__ unsigned long long force_to_fixed(double v) {
    return (unsigned long long)__double2ll_rn(v * FORCE_FIXED_SCALE);
}
__device__ __forceinline__ double force_from_fixed(unsigned long long b) { return (double)(long long)b * FORCE_FIXED_INV; }
template <class P>
__device__ __forceinline__ void force_add(const P& p, size_t idx, double v) {
    if (p.fixed) {
        if (!(fabs(v) < FORCE_FIXED_LIMIT)) {
            atomicOr(p.status, ST_FORCE_RANGE);
            atomicOr(p.sticky, ST_FORCE_RANGE);
            return;
        }
        atomicAdd(reinterpret_cast<unsigned long long*>(p.f_sorted) + idx, force_to_fixed(v));
    } else {
        atomicAdd(p.f_sorted + idx, v);
    }
}
#endif

// ---- launchers (each enqueues on `st`; returns the number of kernels launched) ----------
// skin_mode (neighbour-skin mode, k_sort.cu): 0 off, 1 rebuild forced by the host, 2 the device decides
int launch_sort(const Workspace& w, const Grid& g, int64_t n, int n_elem, const double* d_pos,
                const int32_t* d_type, int skin_mode, double skin, cudaStream_t st);
int launch_neighbors(const Workspace& w, const Grid& g, int64_t n, int n_elem, double rc2, int stride,
                     int max_nbr, int skin_mode, double rs2, int sstride, int smax, cudaStream_t st);
int launch_sf(const Workspace& w, const Grid& g, int64_t n, int n_elem, const ElemProgram* const* d_prog,
              const int* variant, const PassInfo& passes, double rc, int stride, int max_nbr, int g_stride, int na_max,
              int precision, cudaStream_t st);
int launch_mlp(const Workspace& w, int64_t n, int n_elem, int ncell, const NetDesc* nets, int g_stride,
               cudaStream_t st);
int launch_force(const Workspace& w, const Grid& g, int64_t n, int n_elem, const ElemProgram* const* d_prog,
                 const int* variant, const PassInfo& passes, double rc, int stride, int max_nbr, int g_stride, int precision,
                 cudaStream_t st);
// mask words per centre + their prefix (k_sf2.cu); before launch_sf
constexpr int WORD_BUDGET = 320;     // gmask capacity = N * WORD_BUDGET words (a water-like centre with 91 neighbours has 152)
int launch_word_offsets(const Workspace& w, const Grid& g, int64_t n, int n_elem, const ElemProgram* const* d_prog,
                        cudaStream_t st);
// fast path of S2 (lane-owned design, k_sf2.cu): specialised variants only
int launch_sf2(const Workspace& w, const Grid& g, int64_t n, int n_elem, const ElemProgram* const* d_prog,
               const int* variant, const PassInfo& passes, double rc, int stride, int max_nbr, int g_stride, int precision,
               cudaStream_t st);
// fast path of S4 (lane-owned design, k_force2.cu): specialised variants only; f_sorted already zeroed
int launch_force2(const Workspace& w, const Grid& g, int64_t n, int n_elem, const ElemProgram* const* d_prog,
                  const int* variant, const PassInfo& passes, double rc, int stride, int max_nbr, int g_stride, int precision,
                  cudaStream_t st);
// small neighbourhoods (max_neighbors <= 32; k_small.cu): 8 lanes per centre, SpecBase12 elements
int launch_sf_small(const Workspace& w, const Grid& g, int64_t n, int n_elem, const ElemProgram* const* d_prog,
                    const int* variant, double rc, int stride, int max_nbr, int g_stride, bool tiny, cudaStream_t st);
int launch_force_small(const Workspace& w, const Grid& g, int64_t n, int n_elem, const ElemProgram* const* d_prog,
                       const int* variant, double rc, int stride, int max_nbr, int g_stride, bool tiny, int fixed_forces,
                       cudaStream_t st);
int launch_finalize(const Workspace& w, int64_t n, double* d_e_atom, double* d_e_total, double* d_force, int fixed_forces,
                    cudaStream_t st);

// MD loop (k_md.cu)
int launch_vv(int64_t n, int n_elem, const double* h_mass, const int32_t* d_type, const double* d_force, double* d_vel,
              double* d_pos, double dt, bool drift, cudaStream_t st);
// k_noalloc.cu: the kinetic energy with its block sums in a file-scope device array (no workspace, no allocation)
constexpr int64_t NOALLOC_MAX_ATOMS = NNP_NOALLOC_MAX_ATOMS;
constexpr int NOALLOC_MAX_PARTIALS = (int)((NOALLOC_MAX_ATOMS + 255) / 256);        // 16,384 doubles = 128 KB
cudaError_t launch_ekin_noalloc(int64_t n, int n_elem, const double* h_mass, const int32_t* d_type, const double* d_vel,
                                double* d_out, cudaStream_t st, int* launches);
int launch_ekin(int64_t n, int n_elem, const double* h_mass, const int32_t* d_type, const double* d_vel, double* d_part,
                double* d_out, cudaStream_t st);

// exports
int launch_export_counts(const Workspace& w, int64_t n, int n_elem, int32_t* d_counts, cudaStream_t st);
int launch_export_neighbors(const Workspace& w, int64_t n, int n_elem, int stride, const int64_t* d_offsets,
                            int32_t* d_idx, int64_t cap, cudaStream_t st);
int launch_export_rows(const Workspace& w, int64_t n, int g_stride, const double* src_sorted, double* dst,
                       cudaStream_t st);
int launch_scan_i64_from_i32(const int32_t* d_in, int64_t n, int64_t* d_out /* n+1 */, int64_t* d_tmp,
                             cudaStream_t st);
void exclusive_scan_i32(int32_t* d_data, int64_t n, int32_t* d_tmp, cudaStream_t st, int* launches);

size_t mlp_smem_bytes(const NetDesc& net, int ta);

double fp64_peak(int device, double seconds, double* sustained, cudaError_t* err);

}  // namespace nnp

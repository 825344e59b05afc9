// k_small.cu -- S2 / S4 for SMALL neighbourhoods (at most 32 neighbours per atom: the paper's metallic systems, PAPER.md
// L70 / L96: Ni with rc = 3.9 A has 18 neighbours, 153 pairs and 60 contributing triangles per atom).
//
// ncu of the Ni-like workload on the one-warp-per-centre instantiation of k_sf2 / k_force2 (profiles/r1g_metal_ncu.md):
// 2,435 + 2,110 warp-instructions per centre against ~960 ideal, 18 of 32 lanes busy in the staging and radial blocks, two
// triplets per lane -- the per-centre FIXED costs (group table, masks, prefix, seek, reductions over 32 lanes) dominate.
// Here a GROUP OF 8 LANES owns a centre, four centres per warp.  The four groups of a warp step through the same
// warp-uniform loops (trip counts = the warp maximum; a finished or dead group idles), so that every warp-level
// primitive is a plain full-mask one (xor-shuffles of distance 4, 2, 1 stay inside a group; a ballot is cut into the
// four group bytes); their neighbourhoods look alike, so little is lost:
//   * staging, radial block: 18 neighbours over 8 lanes (3 rounds), reductions of 3 shuffle steps;
//   * angular part: the pairs of a pair group are enumerated 8 at a time, tested with the EXACT FP64 predicate
//     c^2 < rc^2 (no FP32 screen, no bit masks), ballot-compacted into a 16-bit (j, k) list in shared memory, and the
//     list is evaluated 8 triplets at a time -- full lanes in the expensive part;
//   * forces: both ends of a triplet go to the centre's shared-memory slot accumulators with shared-memory FP64 atomics
//     (the diagonal-major pair order makes 8 consecutive triplets hit distinct slots almost always); one global FP64 RED
//     per component per neighbour at the end.
// Ni-like workload (1,492,992 atoms): SF 4.66 -> 2.18 ms, force 5.35 -> 3.84 ms, step 12.9 -> 8.9 ms.
// Same formulas, same polynomial special functions (mathfn.cuh) and the same compile-time Specs as k_sf2 / k_force2.
#include "angular.cuh"
#include "geometry.cuh"
#include "stream.cuh"

namespace nnp {

constexpr int SM_SLOTS = 32;                              // neighbour slots per centre: template parameter SLOTS = 32, or 24 for
                                                          // max_neighbors <= 24 (10 instead of 8 resident CTAs of k_force_small)
constexpr int SM_CPW = 4;                                 // centres per warp (8 lanes each)
constexpr int SM_WARPS = 2;                               // warps per CTA
constexpr int SM_CPC = SM_CPW * SM_WARPS;                 // centres per CTA
constexpr int SM_LIST = 120;                              // (j, k) list entries per centre (filled and evaluated in turns)

struct SmallParams {
    int64_t n;
    int n_elem, ncell, stride, g_stride;
    double rc2, k2;                      // k2 = (pi / (2 rc))^2
    double box[3], half[3];
    const double *sx, *sy, *sz;
    const int32_t *cell_start, *nbr, *nbr_cnt;
    double* G;                           // SF kernel: out
    const double* dEdG;                  // force kernel: in
    double* f_sorted;                    // force kernel: accumulated into
    int fixed;                           // 1: fixed-point force accumulation (nnp_internal.h force_add)
    uint16_t* slist;                     // [N][SMALL_LIST_U16] pair lists handed from the SF kernel to the force kernel (or null)
    int32_t *status, *sticky;
    const ElemProgram* prog[MAX_ELEM];
    int variant[MAX_ELEM];
};

// sum of N = 16 per-lane values over the 8 lanes of a group with 8 + 4 + 2 shuffles; afterwards v[0], v[1] of lane gl hold the
// totals of value indices  vi, vi + 1  with  vi = 8 bit2(gl) + 4 bit1(gl) + 2 bit0(gl).  Fixed order: deterministic.
__device__ __forceinline__ void group8_reduce16(double (&v)[16], int gl) {
    {
        const bool hi = (gl & 4) != 0;
#pragma unroll
        for (int t = 0; t < 8; ++t) {
            const double mine = hi ? v[8 + t] : v[t], other = hi ? v[t] : v[8 + t];
            v[t] = mine + __shfl_xor_sync(FULL, other, 4);
        }
    }
    {
        const bool hi = (gl & 2) != 0;
#pragma unroll
        for (int t = 0; t < 4; ++t) {
            const double mine = hi ? v[4 + t] : v[t], other = hi ? v[t] : v[4 + t];
            v[t] = mine + __shfl_xor_sync(FULL, other, 2);
        }
    }
    {
        const bool hi = (gl & 1) != 0;
#pragma unroll
        for (int t = 0; t < 2; ++t) {
            const double mine = hi ? v[2 + t] : v[t], other = hi ? v[t] : v[2 + t];
            v[t] = mine + __shfl_xor_sync(FULL, other, 1);
        }
    }
}

__device__ __forceinline__ double group8_sum(double v) {
    v += __shfl_xor_sync(FULL, v, 4);
    v += __shfl_xor_sync(FULL, v, 2);
    v += __shfl_xor_sync(FULL, v, 1);
    return v;
}

// menu entry (eta slot * 16 + bit) of accumulator index a (inverse of acc_index)
template <class Spec>
__host__ __device__ constexpr int acc_entry(int a) {
    int n = 0;
    for (int e = 0; e < Spec::NETA; ++e)
        for (int b = 0; b < 16; ++b)
            if (Spec::mask(e) >> b & 1u) {
                if (n == a) return e * 16 + b;
                ++n;
            }
    return 0;
}

// Enumerates the pairs of one pair group 8 at a time, keeps those with c^2 < rc^2 (exact FP64 test on the staged
// minimum-image vectors) and writes them as (j << 8 | k) slot pairs to a list of SM_LIST entries in shared memory; the
// caller evaluates the list and calls fill() again until done().  All warp-level primitives of this file take the FULL
// mask and every loop that contains one has a warp-uniform trip count (the four groups of a warp step together; a group
// that is finished, or dead, idles): primitives on four different 8-lane masks per warp were measured far slower
// (k_force_small 7.5 ms with match / vote / syncwarp on group masks).
// Order: DIAGONAL-major -- within a segment all pairs (j, j + r) of r = 1, then r = 2, ...; between two segments
// all pairs (j, (j + r) mod n2) of r = 0, then r = 1, ... -- so that 8 consecutive list entries have pairwise distinct
// j and (almost always) pairwise distinct k: the force kernel's slot updates then rarely wait for each other
// (row-major order put the same j into all 8 lanes of a round: 8 turn-taking passes, 8.9 instead of 5.3 ms).
struct SmallPairs {
    int s1, n1, s2, n2, P;      // segments of the two elements, number of pairs
    bool within;
    int base, r, rem;           // progress: next flattened index = base + gl, at position rem of diagonal r

    __device__ __forceinline__ void start(int s1_, int n1_, int s2_, int n2_, bool within_, int gl) {
        s1 = s1_; n1 = n1_; s2 = s2_; n2 = n2_; within = within_;
        P = within ? n1 * (n1 - 1) / 2 : n1 * n2;
        base = 0; r = within ? 1 : 0; rem = gl;
    }
    __device__ __forceinline__ bool done() const { return base >= P; }

    // appends contributing pairs to list[0 ..) until the pairs are exhausted or fewer than 8 entries of `cap` are free
    __device__ __forceinline__ int fill(const double2* p0, const double2* p1, double rc2, uint16_t* list, int cap, int gl, int grp) {
        int cnt = 0;
        while (true) {
            const bool go = base < P && cnt + 8 <= cap;              // uniform inside the group
            if (!__any_sync(FULL, go)) break;                        // warp-uniform loop: the four groups stay together
            const bool valid = go && base + gl < P;
            int j = 0, k = 0;
            if (valid) {
                if (within) { while (rem >= n1 - r) { rem -= n1 - r; ++r; } j = rem; k = j + r; }
                else { while (rem >= n1) { rem -= n1; ++r; } j = rem; k = j + r; while (k >= n2) k -= n2; }
            }
            const int sj = s1 + j, sk = valid ? (within ? s1 + k : s2 + k) : s1;
            const double2 a0 = p0[sj], a1 = p1[sj], b0 = p0[sk], b1 = p1[sk];
            const double wx = b0.x - a0.x, wy = b0.y - a0.y, wz = b1.x - a1.x;
            const bool pass = valid && fma(wx, wx, fma(wy, wy, wz * wz)) < rc2;
            const unsigned b = (__ballot_sync(FULL, pass) >> (8 * grp)) & 255u;
            if (pass) list[cnt + __popc(b & ((1u << gl) - 1u))] = (uint16_t)((sj << 8) | sk);
            cnt += __popc(b);
            if (go) { rem += 8; base += 8; }
        }
        __syncwarp();
        return cnt;
    }
};

// ---------------------------------------------------------------------------------------------- S2
// shared memory per centre: p0 (ux,uy), p1 (uz,1/a), p2 (exp(-eta0 a^2), fc(a)) double2[32]; ra double[32]; list u16[SM_LIST]
__host__ __device__ constexpr size_t sm_sf_bytes(int slots) { return (size_t)3 * slots * 16 + (size_t)slots * 8 + SM_LIST * 2; }

template <class Spec, bool TINY, int SLOTS>
__global__ void __launch_bounds__(SM_WARPS * 32, 12) k_sf_small(const __grid_constant__ SmallParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NACC = Spec::NACC;
    static_assert(NACC <= 16 && !Spec::FREE_ETA, "k_sf_small: BASELINE.json's 12-function shape (<= 16 accumulators)");
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, grp = lane >> 3, gl = lane & 7;
    const int64_t i0 = (int64_t)blockIdx.x * SM_CPC + wid * SM_CPW + grp;
    const int64_t i = i0 < p.n ? i0 : p.n - 1;
    int tc = 0;
    for (int e = 1; e < p.n_elem; ++e)
        if (i >= p.cell_start[(size_t)e * p.ncell]) tc = e;
    const ElemProgram* __restrict__ prog = p.prog[tc];
    // a group without work (past the end, or an element of another kernel) stays in the warp's loops with empty ranges
    const bool live = i0 < p.n && p.variant[tc] == Spec::ID && (prog->tiny_exp != 0) == TINY;

    unsigned char* base = smem_raw + (size_t)(wid * SM_CPW + grp) * sm_sf_bytes(SLOTS);
    double2* p0 = reinterpret_cast<double2*>(base);
    double2* p1 = p0 + SLOTS;
    double2* p2 = p1 + SLOTS;
    double* ra = reinterpret_cast<double*>(p2 + SLOTS);
    uint16_t* list = reinterpret_cast<uint16_t*>(ra + SLOTS);

    int seg[MAX_ELEM + 1];
    seg[0] = 0;
#pragma unroll
    for (int e = 0; e < MAX_ELEM; ++e) seg[e + 1] = seg[e] + (live ? p.nbr_cnt[(size_t)i * MAX_ELEM + e] : 0);
    const int ntot = seg[MAX_ELEM];

    // ---- stage the neighbourhood
    const double xi = p.sx[i], yi = p.sy[i], zi = p.sz[i];
    const int32_t* row = p.nbr + (size_t)i * p.stride;
    const double eta0 = prog->ang_eta[0];
    // (the <= 4 slots of a lane: all neighbour indices first, then all coordinates -- two round trips instead of eight)
    int jn[SLOTS / 8];
    double xj[SLOTS / 8], yj[SLOTS / 8], zj[SLOTS / 8];
#pragma unroll
    for (int q = 0; q < SLOTS / 8; ++q) jn[q] = gl + 8 * q < ntot ? row[gl + 8 * q] : (int)i;
#pragma unroll
    for (int q = 0; q < SLOTS / 8; ++q) { xj[q] = p.sx[jn[q]]; yj[q] = p.sy[jn[q]]; zj[q] = p.sz[jn[q]]; }
#pragma unroll
    for (int q = 0; q < SLOTS / 8; ++q) {
        const int m = gl + 8 * q;
        if (m >= ntot) continue;
        const double dx = min_image_1d(xi, xj[q], p.box[0], p.half[0]);
        const double dy = min_image_1d(yi, yj[q], p.box[1], p.half[1]);
        const double dz = min_image_1d(zi, zj[q], p.box[2], p.half[2]);
        const double a2 = fma(dx, dx, fma(dy, dy, dz * dz));
        const double ia = rsqrt(a2);
        const double Ca = cos_only(a2 * p.k2);
        p0[m] = make_double2(dx, dy);
        p1[m] = make_double2(dz, ia);
        p2[m] = make_double2(TINY ? exp_tiny(-eta0 * a2) : exp_small(-eta0 * a2), Ca * Ca);
        ra[m] = a2 * ia;
    }
    __syncwarp();
    double* Grow = p.G + (size_t)i * p.g_stride;
    if (live)
        for (int s = prog->n_sf + gl; s < p.g_stride; s += 8) Grow[s] = 0.0;

    // ---- radial: G = sum_j exp(-eta (a - rs)^2) fc(a)
    for (int e = 0; e < p.n_elem; ++e) {
        const int nr = live ? prog->n_rad[e] : 0, off = prog->rad_off[e];
        const int nr_warp = __reduce_max_sync(FULL, nr);
        for (int r = 0; r < nr_warp; ++r) {
            const RadialSF f = prog->rad[off + (r < nr ? r : 0)];
            double acc = 0.0;
            if (r < nr)
                for (int m = seg[e] + gl; m < seg[e + 1]; m += 8) {
                    const double d = ra[m] - f.rs;
                    acc = fma(exp_small(fmax(-f.eta * d * d, -700.0)), p2[m].y, acc);
                }
            acc = group8_sum(acc);
            if (gl == 0 && r < nr) Grow[f.g] = acc;
        }
    }

    // ---- angular: pair group by pair group.  The compacted (j, k) list of a group goes to the force kernel as well (it
    // would enumerate and test the same 153 pairs again: ~16 % of its instructions on the Ni-like workload), if every
    // group of the centre fits one fill and all of them together the per-centre budget; [0] = 0 marks a valid hand-over.
    uint16_t* hlist = (p.slist && live) ? p.slist + (size_t)i * SMALL_LIST_U16 : nullptr;
    bool ho_ok = hlist != nullptr;
    int ho_off = 0;
    for (int e1 = 0; e1 < p.n_elem; ++e1)
        for (int e2 = e1; e2 < p.n_elem; ++e2) {
            const int pr = pair_index(e1, e2, p.n_elem);
            const bool on = live && prog->n_ang[pr] != 0;
            if (hlist && gl == 0) hlist[1 + pr] = 0;
            if (!__any_sync(FULL, on)) continue;
            SmallPairs sp;
            sp.start(seg[e1], on ? seg[e1 + 1] - seg[e1] : 0, seg[e2], on ? seg[e2 + 1] - seg[e2] : 0, e1 == e2, gl);
            double acc[NACC];
#pragma unroll
            for (int a = 0; a < NACC; ++a) acc[a] = 0.0;
            int fills = 0;
            while (__any_sync(FULL, !sp.done())) {
            const bool had_work = !sp.done();
            const int cnt = sp.fill(p0, p1, p.rc2, list, SM_LIST, gl, grp);
            if (had_work) {
                ++fills;
                if (ho_ok && fills == 1 && sp.done() && ho_off + cnt <= SMALL_LIST_U16 - SMALL_LIST_HDR) {
                    for (int t = gl; t < cnt; t += 8) hlist[SMALL_LIST_HDR + ho_off + t] = list[t];
                    if (gl == 0) hlist[1 + pr] = (uint16_t)cnt;
                    ho_off += cnt;
                } else {
                    ho_ok = false;
                }
            }
            for (int t = gl; t < cnt; t += 8) {
                const int jk = list[t], j = jk >> 8, k = jk & 255;
                const double2 a0 = p0[j], a1 = p1[j], a2 = p2[j], k0 = p0[k], k1 = p1[k], k2v = p2[k];
                const double wx = k0.x - a0.x, wy = k0.y - a0.y, wz = k1.x - a1.x;
                const double c2 = fma(wx, wx, fma(wy, wy, wz * wz));
                const double Cc = cos_only(c2 * p.k2);
                const double Cf = (a2.y * k2v.y) * (Cc * Cc);          // fc(a) fc(b) fc(c)
                double Y[Spec::NETA];
                Y[0] = (a2.x * k2v.x) * (TINY ? exp_tiny(-eta0 * c2) : exp_small(-eta0 * c2));
                if constexpr (Spec::NETA > 1) Y[1] = ipow<Spec::ratio(1)>(Y[Spec::rbase(1)]);
                if constexpr (Spec::NETA > 2) Y[2] = ipow<Spec::ratio(2)>(Y[Spec::rbase(2)]);
                if constexpr (Spec::NETA > 3) Y[3] = ipow<Spec::ratio(3)>(Y[Spec::rbase(3)]);
                const double cosv = fma(a0.x, k0.x, fma(a0.y, k0.y, a1.x * k1.x)) * (a1.y * k1.y);
                double pw[2][Spec::MAXBIT + 1];
                pw[0][0] = 1.0 + cosv;
                pw[1][0] = 1.0 - cosv;
#pragma unroll
                for (int b = 1; b <= Spec::MAXBIT; ++b) {
                    pw[0][b] = pw[0][b - 1] * pw[0][b - 1];
                    pw[1][b] = pw[1][b - 1] * pw[1][b - 1];
                }
#pragma unroll
                for (int e = 0; e < Spec::NETA; ++e) {
                    const double xc = Y[e] * Cf;
#pragma unroll
                    for (int b = 0; b <= Spec::MAXBIT; ++b) {
                        if (Spec::mask(e) >> b & 1u) acc[acc_index<Spec>(e, b)] = fma(pw[0][b], xc, acc[acc_index<Spec>(e, b)]);
                        if (Spec::mask(e) >> (8 + b) & 1u)
                            acc[acc_index<Spec>(e, 8 + b)] = fma(pw[1][b], xc, acc[acc_index<Spec>(e, 8 + b)]);
                    }
                }
            }
            __syncwarp();                              // the list is refilled
            }
            double v[16];
#pragma unroll
            for (int a = 0; a < 16; ++a) v[a] = a < NACC ? acc[a < NACC ? a : 0] : 0.0;
            group8_reduce16(v, gl);
            const int vi = ((gl & 4) ? 8 : 0) + ((gl & 2) ? 4 : 0) + ((gl & 1) ? 2 : 0);
#pragma unroll
            for (int a = 0; a < NACC; ++a) {
                if (on && (a == vi || a == vi + 1)) {
                    const int en = acc_entry<Spec>(a), e = en >> 4, b = en & 15;
                    const int g = prog->ang_g[pr][e][b];
                    if (g >= 0) Grow[g] = exp2((double)(1 - (1 << (b & 7)))) * (a == vi ? v[0] : v[1]);
                }
            }
            __syncwarp();                              // the list is reused by the next pair group
        }
    if (hlist && gl == 0) hlist[0] = ho_ok ? 0 : 1;
}

// ---------------------------------------------------------------------------------------------- S4
// shared memory per centre: p0 (ux,uy), p1 (uz,1/a), p2 (fc(a), fc'(a)/a) double2[32]; e0, rad, fx, fy, fz double[32];
// beta row double[g_stride]; coefficients c_b = beta_b 2^(1-zeta_b) double[npair][16]; list u16[SM_LIST]
__host__ __device__ constexpr size_t sm_force_bytes(int g_stride, int n_elem, int slots) {
    return (size_t)3 * slots * 16 + (size_t)5 * slots * 8 + (size_t)((g_stride + 1) & ~1) * 8 +
           (size_t)(n_elem * (n_elem + 1) / 2) * 16 * 8 + SM_LIST * 2;
}

// acc[slot] += v for the lanes with act.  Shared-memory FP64 atomics (a compare-and-swap loop on sm_100a): in the big
// kernels they lost to turn-taking (2.9 lanes per slot and iteration), here 8 consecutive list entries hit distinct
// slots almost always, the CAS succeeds at once, and no warp-synchronous instruction (match / vote / syncwarp on a
// group mask: four masks per warp) is left in the triplet loop -- 5.4 instead of 7.5 ms on the Ni-like workload.
__device__ __forceinline__ void small_slot_add(double* fx, double* fy, double* fz, int slot, bool act, double x, double y, double z,
                                               int fixed) {
    if (!act) return;
    if (fixed) {            // deterministic mode: 64-bit integer adds (native shared-memory atomics, any order gives the same bits)
        atomicAdd(reinterpret_cast<unsigned long long*>(fx) + slot, force_to_fixed(x));
        atomicAdd(reinterpret_cast<unsigned long long*>(fy) + slot, force_to_fixed(y));
        atomicAdd(reinterpret_cast<unsigned long long*>(fz) + slot, force_to_fixed(z));
    } else {
        atomicAdd(&fx[slot], x);
        atomicAdd(&fy[slot], y);
        atomicAdd(&fz[slot], z);
    }
}

template <class Spec, bool TINY, int SLOTS>
__global__ void __launch_bounds__(SM_WARPS * 32, SLOTS <= 24 ? 10 : 8) k_force_small(const __grid_constant__ SmallParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NACC = Spec::NACC;
    static_assert(NACC <= 16 && !Spec::FREE_ETA, "k_force_small: BASELINE.json's 12-function shape (<= 16 accumulators)");
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, grp = lane >> 3, gl = lane & 7;
    const int64_t i0 = (int64_t)blockIdx.x * SM_CPC + wid * SM_CPW + grp;
    const int64_t i = i0 < p.n ? i0 : p.n - 1;
    int tc = 0;
    for (int e = 1; e < p.n_elem; ++e)
        if (i >= p.cell_start[(size_t)e * p.ncell]) tc = e;
    const ElemProgram* __restrict__ prog = p.prog[tc];
    // a group without work (past the end, or an element of another kernel) stays in the warp's loops with empty ranges
    const bool live = i0 < p.n && p.variant[tc] == Spec::ID && (prog->tiny_exp != 0) == TINY;

    const int npair = p.n_elem * (p.n_elem + 1) / 2;
    unsigned char* base = smem_raw + (size_t)(wid * SM_CPW + grp) * sm_force_bytes(p.g_stride, p.n_elem, SLOTS);
    double2* p0 = reinterpret_cast<double2*>(base);
    double2* p1 = p0 + SLOTS;
    double2* p2 = p1 + SLOTS;
    double* e0 = reinterpret_cast<double*>(p2 + SLOTS);
    double* rad = e0 + SLOTS;
    double* fx = rad + SLOTS;
    double* fy = fx + SLOTS;
    double* fz = fy + SLOTS;
    double* brow = fz + SLOTS;
    double* cft = brow + ((p.g_stride + 1) & ~1);
    uint16_t* list = reinterpret_cast<uint16_t*>(cft + npair * 16);

    int seg[MAX_ELEM + 1];
    seg[0] = 0;
#pragma unroll
    for (int e = 0; e < MAX_ELEM; ++e) seg[e + 1] = seg[e] + (live ? p.nbr_cnt[(size_t)i * MAX_ELEM + e] : 0);
    const int ntot = seg[MAX_ELEM];

    for (int s = gl; s < p.g_stride; s += 8) brow[s] = live ? p.dEdG[(size_t)i * p.g_stride + s] : 0.0;
    __syncwarp();

    // ---- stage the neighbourhood; radial part R = sum_r beta_r exp(-eta d^2) (fc'(a) - 2 eta d fc(a)) / a
    const double xi = p.sx[i], yi = p.sy[i], zi = p.sz[i];
    const int32_t* row = p.nbr + (size_t)i * p.stride;
    const double eta0 = prog->ang_eta[0];
    int jn[SLOTS / 8];
    double xj[SLOTS / 8], yj[SLOTS / 8], zj[SLOTS / 8];
#pragma unroll
    for (int q = 0; q < SLOTS / 8; ++q) jn[q] = gl + 8 * q < ntot ? row[gl + 8 * q] : (int)i;
#pragma unroll
    for (int q = 0; q < SLOTS / 8; ++q) { xj[q] = p.sx[jn[q]]; yj[q] = p.sy[jn[q]]; zj[q] = p.sz[jn[q]]; }
#pragma unroll
    for (int q = 0; q < SLOTS / 8; ++q) {
        const int m = gl + 8 * q;
        if (m >= ntot) continue;
        int e = 0;                                           // element of slot m
        for (int t = 1; t < p.n_elem; ++t)
            if (m >= seg[t]) e = t;
        const int nr = prog->n_rad[e], off = prog->rad_off[e];
        {
            const double dx = min_image_1d(xi, xj[q], p.box[0], p.half[0]);
            const double dy = min_image_1d(yi, yj[q], p.box[1], p.half[1]);
            const double dz = min_image_1d(zi, zj[q], p.box[2], p.half[2]);
            const double a2 = fma(dx, dx, fma(dy, dy, dz * dz));
            const double ia = rsqrt(a2);
            const double a = a2 * ia;
            double Ca, Sa;
            cos_sinc(a2 * p.k2, Ca, Sa);
            const double fa = Ca * Ca;
            const double dfa_a = (-2.0 * p.k2) * (Ca * Sa);
            p0[m] = make_double2(dx, dy);
            p1[m] = make_double2(dz, ia);
            p2[m] = make_double2(fa, dfa_a);
            e0[m] = TINY ? exp_tiny(-eta0 * a2) : exp_small(-eta0 * a2);
            double Rs = 0.0;
            for (int r = 0; r < nr; ++r) {
                const RadialSF f = prog->rad[off + r];
                const double d = a - f.rs;
                const double ex = exp_small(fmax(-f.eta * d * d, -700.0));
                Rs = fma(brow[f.g] * ex, fma(-2.0 * f.eta * d, fa * ia, dfa_a), Rs);
            }
            rad[m] = Rs;
            fx[m] = 0.0; fy[m] = 0.0; fz[m] = 0.0;
        }
    }
    // coefficients of all pair groups: c_a = beta_g(a) 2^(1 - zeta(a))
    for (int s = gl; s < npair * 16; s += 8) {
        const int pr = s >> 4, a = s & 15;
        double c = 0.0;
#pragma unroll
        for (int q = 0; q < NACC; ++q)
            if (q == a) {
                const int en = acc_entry<Spec>(q), e = en >> 4, b = en & 15;
                const int g = prog->ang_g[pr][e][b];
                if (g >= 0) c = brow[g] * exp2((double)(1 - (1 << (b & 7))));
            }
        cft[s] = c;
    }
    __syncwarp();

    double eta[Spec::NETA];
#pragma unroll
    for (int e = 0; e < Spec::NETA; ++e) eta[e] = prog->ang_eta[e];

    // the pair lists of the symmetry-function kernel, if it handed them over for this centre (k_sf_small)
    const uint16_t* hlist = (p.slist && live) ? p.slist + (size_t)i * SMALL_LIST_U16 : nullptr;
    const bool use_ho = hlist != nullptr && hlist[0] == 0;
    int ho_off = 0;

    // ---- angular part: pair group by pair group
    for (int e1 = 0; e1 < p.n_elem; ++e1)
        for (int e2 = e1; e2 < p.n_elem; ++e2) {
            const int pr = pair_index(e1, e2, p.n_elem);
            const bool on = live && prog->n_ang[pr] != 0;
            if (!__any_sync(FULL, on)) continue;
            // a centre whose lists came from the SF kernel enumerates nothing (empty ranges: it idles through fill())
            const bool mine = on && !use_ho;
            SmallPairs sp;
            sp.start(seg[e1], mine ? seg[e1 + 1] - seg[e1] : 0, seg[e2], mine ? seg[e2 + 1] - seg[e2] : 0, e1 == e2, gl);
            const int hc = (on && use_ho) ? (int)hlist[1 + pr] : 0;
            bool pend = hc > 0;
            double cf[NACC];
#pragma unroll
            for (int a = 0; a < NACC; ++a) cf[a] = cft[pr * 16 + a];
            while (__any_sync(FULL, !sp.done() || pend)) {
            int cnt = sp.fill(p0, p1, p.rc2, list, SM_LIST, gl, grp);
            if (pend) {
                for (int t = gl; t < hc; t += 8) list[t] = hlist[SMALL_LIST_HDR + ho_off + t];
                cnt = hc;
                ho_off += hc;
                pend = false;
            }
            __syncwarp();
            const int rounds = (cnt + 7) >> 3;
            for (int q = 0; q < rounds; ++q) {
                const int t = q * 8 + gl;
                const bool active = t < cnt;
                const int jk = active ? list[t] : ((seg[e1] << 8) | seg[e1]);
                const int j = jk >> 8, k = jk & 255;
                const double2 a0 = p0[j], a1 = p1[j], a2v = p2[j], k0 = p0[k], k1 = p1[k], k2v = p2[k];
                const double ej = e0[j], ek = e0[k];
                const double wx = k0.x - a0.x, wy = k0.y - a0.y, wz = k1.x - a1.x;
                const double c2 = fma(wx, wx, fma(wy, wy, wz * wz));
                double Cc, Sc;
                cos_sinc(c2 * p.k2, Cc, Sc);
                double fcc = Cc * Cc;                          // fc(c)
                double dfc = (-2.0 * p.k2) * (Cc * Sc);        // fc'(c)/c
                if (!active) { fcc = 0.0; dfc = 0.0; }
                double Y[Spec::NETA];
                Y[0] = (ej * ek) * (TINY ? exp_tiny(-eta0 * c2) : exp_small(-eta0 * c2));
                if constexpr (Spec::NETA > 1) Y[1] = ipow<Spec::ratio(1)>(Y[Spec::rbase(1)]);
                if constexpr (Spec::NETA > 2) Y[2] = ipow<Spec::ratio(2)>(Y[Spec::rbase(2)]);
                if constexpr (Spec::NETA > 3) Y[3] = ipow<Spec::ratio(3)>(Y[Spec::rbase(3)]);
                const double iab = a1.y * k1.y;
                const double cosv = fma(a0.x, k0.x, fma(a0.y, k0.y, a1.x * k1.x)) * iab;
                // pw[l][b] = (1 +- cos)^(2^b) ; pd[l][b] = 2^b (1 +- cos)^(2^b - 1)
                double pw[2][Spec::MAXBIT + 1], pd[2][Spec::MAXBIT + 1];
                pw[0][0] = 1.0 + cosv; pw[1][0] = 1.0 - cosv;
                pd[0][0] = 1.0; pd[1][0] = 1.0;
#pragma unroll
                for (int b = 1; b <= Spec::MAXBIT; ++b) {
#pragma unroll
                    for (int l = 0; l < 2; ++l) {
                        pw[l][b] = pw[l][b - 1] * pw[l][b - 1];
                        pd[l][b] = (2.0 * pd[l][b - 1]) * pw[l][b - 1];
                    }
                }
                double Z0 = 0.0, Z1 = 0.0, Z2 = 0.0;
#pragma unroll
                for (int e = 0; e < Spec::NETA; ++e) {
                    double T0 = 0.0, T1 = 0.0;
#pragma unroll
                    for (int b = 0; b <= Spec::MAXBIT; ++b) {
#pragma unroll
                        for (int l = 0; l < 2; ++l)
                            if (Spec::mask(e) >> (8 * l + b) & 1u) {
                                const double c = cf[acc_index<Spec>(e, 8 * l + b)];
                                T0 = fma(c, pw[l][b], T0);
                                T1 = l == 0 ? fma(c, pd[l][b], T1) : fma(-c, pd[l][b], T1);
                            }
                    }
                    const double A = T0 * Y[e];
                    Z0 += A;
                    Z1 = fma(T1, Y[e], Z1);
                    Z2 = fma(eta[e], A, Z2);
                }
                const double fab = a2v.x * k2v.x;
                const double Cf = fab * fcc;
                const double t2 = (Cf + Cf) * Z2;
                const double f_w = fma(fab * dfc, Z0, -t2);
                const double qq = Z1 * Cf;
                const double qc = qq * cosv;
                const double f_uu = fma(-qc, a1.y * a1.y, fma((a2v.y * k2v.x) * fcc, Z0, -t2));
                const double f_vv = fma(-qc, k1.y * k1.y, fma((a2v.x * k2v.y) * fcc, Z0, -t2));
                const double s1 = f_uu + f_w, s2 = f_vv + f_w, s3 = fma(-qq, iab, f_w);
                // F_j = s3 v - s1 u ,  F_k = s3 u - s2 v
                small_slot_add(fx, fy, fz, j, active, fma(s3, k0.x, -s1 * a0.x), fma(s3, k0.y, -s1 * a0.y), fma(s3, k1.x, -s1 * a1.x), p.fixed);
                small_slot_add(fx, fy, fz, k, active, fma(s3, a0.x, -s2 * k0.x), fma(s3, a0.y, -s2 * k0.y), fma(s3, a1.x, -s2 * k1.x), p.fixed);
            }
            __syncwarp();                              // the list is refilled
            }
        }

    // ---- flush: F_slot - R u; one global FP64 RED per component per neighbour; the centre gets minus the sum
    double sx_ = 0.0, sy_ = 0.0, sz_ = 0.0;
    for (int m = gl; m < ntot; m += 8) {
        const int j = row[m];
        const double2 u0 = p0[m];
        const double uz = p1[m].x, R = rad[m];
        const double gx = p.fixed ? force_from_fixed(reinterpret_cast<const unsigned long long*>(fx)[m]) : fx[m];
        const double gy = p.fixed ? force_from_fixed(reinterpret_cast<const unsigned long long*>(fy)[m]) : fy[m];
        const double gz = p.fixed ? force_from_fixed(reinterpret_cast<const unsigned long long*>(fz)[m]) : fz[m];
        const double ax = fma(-R, u0.x, gx), ay = fma(-R, u0.y, gy), az = fma(-R, uz, gz);
        force_add(p, 3 * (size_t)j + 0, ax);
        force_add(p, 3 * (size_t)j + 1, ay);
        force_add(p, 3 * (size_t)j + 2, az);
        sx_ -= ax; sy_ -= ay; sz_ -= az;
    }
    sx_ = group8_sum(sx_); sy_ = group8_sum(sy_); sz_ = group8_sum(sz_);
    if (gl == 0 && live) {
        force_add(p, 3 * (size_t)i + 0, sx_);
        force_add(p, 3 * (size_t)i + 1, sy_);
        force_add(p, 3 * (size_t)i + 2, sz_);
    }
}

// ---------------------------------------------------------------------------------------------- launchers
static SmallParams small_params(const Workspace& w, const Grid& g, int64_t n, int n_elem, const ElemProgram* const* d_prog,
                                const int* variant, double rc, int stride, int g_stride) {
    SmallParams p;
    p.n = n; p.n_elem = n_elem; p.ncell = g.ncell; p.stride = stride; p.g_stride = g_stride;
    p.rc2 = rc * rc;
    p.k2 = (3.14159265358979323846 / (2.0 * rc)) * (3.14159265358979323846 / (2.0 * rc));
    for (int c = 0; c < 3; ++c) { p.box[c] = g.box[c]; p.half[c] = g.half[c]; }
    p.sx = w.sx; p.sy = w.sy; p.sz = w.sz;
    p.cell_start = w.cell_start; p.nbr = w.nbr; p.nbr_cnt = w.nbr_cnt;
    p.G = w.G; p.dEdG = w.dEdG; p.f_sorted = w.f_sorted;
    p.fixed = 0; p.status = w.status; p.sticky = w.sticky; p.slist = w.slist;
    for (int e = 0; e < MAX_ELEM; ++e) {
        p.prog[e] = e < n_elem ? d_prog[e] : nullptr;
        p.variant[e] = e < n_elem ? (variant[e] & 255) : -1;
    }
    return p;
}

// SpecBase12 elements with max_neighbors <= 32; tiny = the element's exp variant (bit 8 of variant[]); 24 neighbour slots per
// centre if max_neighbors <= 24 (rows never hold more than max_neighbors entries), else 32
template <int SLOTS>
static void launch_sf_small_slots(const SmallParams& p, unsigned grid, bool tiny, cudaStream_t st) {
    const size_t smem = SM_CPC * sm_sf_bytes(SLOTS);
    if (tiny) k_sf_small<SpecBase12, true, SLOTS><<<grid, SM_WARPS * 32, smem, st>>>(p);
    else k_sf_small<SpecBase12, false, SLOTS><<<grid, SM_WARPS * 32, smem, st>>>(p);
}

int launch_sf_small(const Workspace& w, const Grid& g, int64_t n, int n_elem, const ElemProgram* const* d_prog,
                    const int* variant, double rc, int stride, int max_nbr, int g_stride, bool tiny, cudaStream_t st) {
    if (n == 0) return 0;
    const SmallParams p = small_params(w, g, n, n_elem, d_prog, variant, rc, stride, g_stride);
    const unsigned grid = (unsigned)((n + SM_CPC - 1) / SM_CPC);
    if (max_nbr <= 24) launch_sf_small_slots<24>(p, grid, tiny, st);
    else launch_sf_small_slots<32>(p, grid, tiny, st);
    return 1;
}

template <int SLOTS>
static void launch_force_small_slots(const SmallParams& p, unsigned grid, bool tiny, cudaStream_t st) {
    const size_t smem = SM_CPC * sm_force_bytes(p.g_stride, p.n_elem, SLOTS);
    static unsigned long long c1 = 0ull, c0 = 0ull;      // per device and instantiation (opt_in_smem): > 48 KB with wide G rows
    if (tiny) {
        opt_in_smem(k_force_small<SpecBase12, true, SLOTS>, &c1);
        k_force_small<SpecBase12, true, SLOTS><<<grid, SM_WARPS * 32, smem, st>>>(p);
    } else {
        opt_in_smem(k_force_small<SpecBase12, false, SLOTS>, &c0);
        k_force_small<SpecBase12, false, SLOTS><<<grid, SM_WARPS * 32, smem, st>>>(p);
    }
}

int launch_force_small(const Workspace& w, const Grid& g, int64_t n, int n_elem, const ElemProgram* const* d_prog,
                       const int* variant, double rc, int stride, int max_nbr, int g_stride, bool tiny, int fixed_forces,
                       cudaStream_t st) {
    if (n == 0) return 0;
    SmallParams p = small_params(w, g, n, n_elem, d_prog, variant, rc, stride, g_stride);
    p.fixed = fixed_forces;
    const unsigned grid = (unsigned)((n + SM_CPC - 1) / SM_CPC);
    if (max_nbr <= 24) launch_force_small_slots<24>(p, grid, tiny, st);
    else launch_force_small_slots<32>(p, grid, tiny, st);
    return 1;
}

}  // namespace nnp

// angular.cuh -- pieces shared by the symmetry-function kernel (k_sf.cu) and the force kernel
// (k_force.cu): compile-time descriptions of angular pair groups, per-warp shared-memory
// layout of a centre's neighbourhood, and the triplet enumeration with warp compaction.
//
// Design: one warp owns one centre atom.  Its neighbours are staged once
// in shared memory (min-image vectors, 1/r, cutoff values, per-eta Gaussians); candidate
// (j,k) pairs are enumerated in rounds (round r pairs slot j with slot j+r), the cheap
// r_jk < rc test is ballot-compacted into a small FIFO, and the expensive per-triplet work
// runs only on full batches of 32 contributing triplets -> no idle lanes in the hot loop
// even though only ~47 % of the enumerated pairs contribute.
#pragma once
#include "mathfn.cuh"
#include "nnp_internal.h"

namespace nnp {

// ---------------------------------------------------------------- compile-time group specs
// A specialised group is: NETA distinct etas with eta_e = eta_{RBASE(e)} * RATIO(e) (integer
// ratios -> exp(-eta_e x) is a short multiplication chain of exp(-eta_0 x)), and per eta a
// bit mask of (lambda, zeta) menu entries: bit b (0..6) = lambda +1, zeta 2^b; bit 8+b =
// lambda -1, zeta 2^b.

struct SpecGeneric {
    static constexpr int ID = ANG_GENERIC;
    static constexpr int NETA = 0;
    static constexpr int MAXBIT = 0;
    static constexpr int NACC = 0;
    static constexpr bool FREE_ETA = false;
    __host__ __device__ static constexpr unsigned mask(int) { return 0u; }
    __host__ __device__ static constexpr int ratio(int) { return 1; }
    __host__ __device__ static constexpr int rbase(int) { return 0; }
};

// BASELINE.json base set (reading C8): eta0 x {+-1} x {1,2,4,16}  +  10*eta0 x {+1} x {1,2,4,16}
struct SpecBase12 {
    static constexpr int ID = ANG_BASE12;
    static constexpr int NETA = 2;
    static constexpr int MAXBIT = 4;
    static constexpr int NACC = 12;
    static constexpr bool FREE_ETA = false;
    __host__ __device__ static constexpr unsigned mask(int e) { return e == 0 ? 0x1717u : (e == 1 ? 0x0017u : 0u); }
    __host__ __device__ static constexpr int ratio(int e) { return e == 1 ? 10 : 1; }
    __host__ __device__ static constexpr int rbase(int) { return 0; }
};

// wide set (reading C9): eta0 x {1,3,10,30}, each x {+-1} x {1,2,4,16}
struct SpecWide32 {
    static constexpr int ID = ANG_WIDE32;
    static constexpr int NETA = 4;
    static constexpr int MAXBIT = 4;
    static constexpr int NACC = 32;
    static constexpr bool FREE_ETA = false;
    __host__ __device__ static constexpr unsigned mask(int e) { return e < 4 ? 0x1717u : 0u; }
    __host__ __device__ static constexpr int ratio(int e) { return e == 1 ? 3 : (e == 2 ? 10 : (e == 3 ? 3 : 1)); }
    __host__ __device__ static constexpr int rbase(int e) { return e == 3 ? 2 : 0; }
};

// Any table with at most four distinct eta values (no ratio between them), lambda = +-1 and zeta in {1,2,4,16}: the
// menu of SpecWide32 with entries allowed to be missing (coefficient 0 / no G index) and exp(-eta_e r^2) evaluated
// per eta instead of as an integer power of the first -- the lane-owned kernels for models that are not BASELINE.json's.
struct SpecFree32 {
    static constexpr int ID = ANG_FREE32;
    static constexpr int NETA = 4;
    static constexpr int MAXBIT = 4;
    static constexpr int NACC = 32;
    static constexpr bool FREE_ETA = true;
    __host__ __device__ static constexpr unsigned mask(int e) { return e < 4 ? 0x1717u : 0u; }
    __host__ __device__ static constexpr int ratio(int) { return 1; }
    __host__ __device__ static constexpr int rbase(int) { return 0; }
};

// the same for tables with one or two eta values: half the accumulators, more resident CTAs
struct SpecFree16 {
    static constexpr int ID = ANG_FREE16;
    static constexpr int NETA = 2;
    static constexpr int MAXBIT = 4;
    static constexpr int NACC = 16;
    static constexpr bool FREE_ETA = true;
    __host__ __device__ static constexpr unsigned mask(int e) { return e < 2 ? 0x1717u : 0u; }
    __host__ __device__ static constexpr int ratio(int) { return 1; }
    __host__ __device__ static constexpr int rbase(int) { return 0; }
};

// accumulator slot of menu entry (e, bit) = number of set menu bits before it
template <class Spec>
__host__ __device__ constexpr int acc_index(int e, int bit) {
    int n = 0;
    for (int ee = 0; ee < Spec::NETA; ++ee)
        for (int b = 0; b < 16; ++b) {
            if (ee == e && b == bit) return n;
            if (Spec::mask(ee) >> b & 1u) ++n;
        }
    return n;
}

template <int K>
__device__ __forceinline__ double ipow(double x) {
    if constexpr (K <= 1) return x;
    else if constexpr (K % 2 == 0) { const double h = ipow<K / 2>(x); return h * h; }
    else return x * ipow<K - 1>(x);
}

// E[e] = exp(-eta_e * x) for all etas of the spec from ONE exp() and multiplication chains
template <class Spec>
__device__ __forceinline__ void eta_chain(double x, double eta0, double* E) {
    E[0] = exp_small(-eta0 * x);    // nnp_create admits a Spec only if eta_max * 3 rc^2 <= 700
    if constexpr (Spec::NETA > 1) E[1] = ipow<Spec::ratio(1)>(E[Spec::rbase(1)]);
    if constexpr (Spec::NETA > 2) E[2] = ipow<Spec::ratio(2)>(E[Spec::rbase(2)]);
    if constexpr (Spec::NETA > 3) E[3] = ipow<Spec::ratio(3)>(E[Spec::rbase(3)]);
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}

// Sum N (power of two, <= 32) per-lane values over the warp with N - 1 + log2(32 / N) 64-bit shuffles
// instead of 5 N: at every step a lane keeps one half of its values and hands the other half to its
// partner.  On return s[0] of lane l holds the total of value index  vi = sum_t bit_(4-t)(l) * (N >> (t+1))
// (warp_reduce_index), in every lane of the group that shares those bits.  Fixed order -> deterministic.
template <int N>
__device__ __forceinline__ void warp_reduce_multi(double (&s)[N], int lane) {
    static_assert(N == 1 || N == 2 || N == 4 || N == 8 || N == 16 || N == 32, "N must be a power of two");
    int width = N, delta = 16;
#pragma unroll
    for (int step = 0; step < 5; ++step) {
        if (width > 1) {
            const int half = width >> 1;
            const bool hi = (lane & delta) != 0;
#pragma unroll
            for (int t = 0; t < N / 2; ++t) {
                if (t < half) {
                    const double mine = hi ? s[half + t] : s[t];
                    const double other = hi ? s[t] : s[half + t];
                    s[t] = mine + __shfl_xor_sync(0xffffffffu, other, delta);
                }
            }
            width = half;
        } else {
            s[0] += __shfl_xor_sync(0xffffffffu, s[0], delta);
        }
        delta >>= 1;
    }
}

template <int N>
__device__ __forceinline__ int warp_reduce_index(int lane) {
    int vi = 0, width = N, delta = 16;
#pragma unroll
    for (int step = 0; step < 5; ++step) {
        if (width > 1) {
            width >>= 1;
            if (lane & delta) vi += width;
        }
        delta >>= 1;
    }
    return vi;
}

// ---------------------------------------------------------------- per-warp neighbourhood in smem
// Slot m (0..n-1) of the centre's neighbour row, grouped by element.  Packed as double2 so the
// per-triplet gathers are 128-bit shared loads.  A second, FP32 copy of the min-image vectors
// feeds the candidate screening (below): 12 B per slot instead of 24 B, FP32 pipe instead of FP64.
struct Nbh {
    double2* p0;   // (ux, uy)
    double2* p1;   // (uz, 1/a)
    double2* p2;   // SF kernel: (exp(-eta_0 a^2), fc(a));  force kernel: (fc(a), fc'(a)/a)
                   // fc(a) = C^2, fc'(a)/a = -2 k2 C S with z = k2 a^2, k2 = (pi/(2 rc))^2 (mathfn.cuh)
    double2* p3;   // force kernel only: (exp(-eta_0 a^2), unused)
    float2* fxy;   // (float ux, float uy)
    float* fz;     // float uz
};

// ---------------------------------------------------------------- triplet enumeration
// Calls f(j, k, colour, active) for batches of 32 candidate pairs that passed the SCREEN
//     |u_k - u_j|^2 < rc^2 (1 + 1e-5)      evaluated in FP32 on the FP32 copies
// (FP32 error of that expression is < 1e-6 rc^2, so no contributing pair is ever dropped); the
// functor applies the exact FP64 test c^2 < rc^2 itself and zeroes fc(c) otherwise.  ncu on the first
// version (profiles/r1_k_force_k_sf_summary.md) showed the FP64 pair test with four shared loads per
// candidate to be 35 % of the instructions and 20 % of the shared-memory wavefronts of k_force.
//
// Pairs are visited in ROUNDS flattened into one index p so that all 32 lanes stay busy: within
// a segment of ns slots, p = (r-1) ns + j pairs slot j with slot (j + r) mod ns, r = 1..ns/2 (the
// last round of an even ns is half) -- inside one round every slot appears at most once as j and
// at most once as k.  Between two segments, p = r n_small + s pairs slot s of the smaller segment
// with slot (s + r) mod n_big of the bigger one.  The round number travels with the pair through
// the compaction queue as its COLOUR: entries of equal colour never share a j or a k, which lets
// the force kernel accumulate per-slot forces with plain shared-memory read-modify-writes, one
// colour at a time, instead of FP64 shared atomics (CAS loops).  The queue is a 64-entry FIFO
// ring per warp.
struct PairQueue {
    uint32_t* q;    // [64] (colour << 16) | (j << 8) | k
    int head, n;
};

__device__ __forceinline__ void q_push(PairQueue& Q, bool pass, int j, int k, int col, int lane) {
    const unsigned m = __ballot_sync(0xffffffffu, pass);
    if (pass) Q.q[(Q.head + Q.n + __popc(m & ((1u << lane) - 1u))) & 63] = ((unsigned)col << 16) | (unsigned)((j << 8) | k);
    Q.n += __popc(m);
    __syncwarp();
}

// pop min(32, n) entries (n >= 1) and hand them to f; idle lanes replay entry 0 with active = false
template <class F>
__device__ __forceinline__ void q_pop(PairQueue& Q, int lane, F& f) {
    const int cnt = Q.n < 32 ? Q.n : 32;
    const bool act = lane < cnt;
    const unsigned e = Q.q[(Q.head + (act ? lane : 0)) & 63];
    Q.head = (Q.head + cnt) & 63;
    Q.n -= cnt;
    __syncwarp();
    f((int)((e >> 8) & 255u), (int)(e & 255u), (int)(e >> 16), act);
}

__device__ __forceinline__ bool pair_close32(const Nbh& nb, int j, int k, float rc2f) {
    const float2 a = nb.fxy[j], b = nb.fxy[k];
    const float wx = b.x - a.x, wy = b.y - a.y, wz = nb.fz[k] - nb.fz[j];
    return fmaf(wx, wx, fmaf(wy, wy, wz * wz)) < rc2f;
}

// all unordered pairs inside segment [s, s+ns); colours 1..ns/2; the queue is empty on return
template <class F>
__device__ __forceinline__ void pairs_within(const Nbh& nb, int s, int ns, float rc2f, PairQueue& Q, int lane, F& f) {
    const int P = ns * (ns - 1) / 2;
    if (P <= 0) return;
    int jj = lane, r = 1;
    while (jj >= ns) { jj -= ns; ++r; }
    int p0 = 0;
    while (true) {
        if (p0 < P) {
            bool pass = false;
            int kk = jj + r;
            if (p0 + lane < P) {                    // r <= ns/2 here, so one wrap is enough
                if (kk >= ns) kk -= ns;
                pass = pair_close32(nb, s + jj, s + kk, rc2f);
            }
            q_push(Q, pass, s + jj, s + kk, r, lane);
            p0 += 32;
            jj += 32;
            while (jj >= ns) { jj -= ns; ++r; }
        }
        if (Q.n >= 32 || (p0 >= P && Q.n > 0)) q_pop(Q, lane, f);
        else if (p0 >= P) break;
    }
}

// all pairs (j in [s1, s1+n1), k in [s2, s2+n2)), disjoint segments; colours 0..max(n1,n2)-1
template <class F>
__device__ __forceinline__ void pairs_between(const Nbh& nb, int s1, int n1, int s2, int n2, float rc2f, PairQueue& Q,
                                              int lane, F& f) {
    if (n1 == 0 || n2 == 0) return;
    const bool swap = n1 < n2;                 // the fast index walks the smaller segment
    const int ss = swap ? s1 : s2, ns = swap ? n1 : n2;      // small
    const int sb = swap ? s2 : s1, nbig = swap ? n2 : n1;    // big
    const int P = ns * nbig;
    int qs = lane, r = 0;
    while (qs >= ns) { qs -= ns; ++r; }
    int p0 = 0;
    while (true) {
        if (p0 < P) {
            bool pass = false;
            int qb = qs + r, j = 0, k = 0;
            if (p0 + lane < P) {                    // r < nbig and qs < ns <= nbig: one wrap is enough
                if (qb >= nbig) qb -= nbig;
                j = swap ? ss + qs : sb + qb;       // j from segment 1, k from segment 2
                k = swap ? sb + qb : ss + qs;
                pass = pair_close32(nb, j, k, rc2f);
            }
            q_push(Q, pass, j, k, r, lane);
            p0 += 32;
            qs += 32;
            while (qs >= ns) { qs -= ns; ++r; }
        }
        if (Q.n >= 32 || (p0 >= P && Q.n > 0)) q_pop(Q, lane, f);
        else if (p0 >= P) break;
    }
}

// screening threshold (see above)
__device__ __forceinline__ float screen_rc2(double rc2) { return (float)(rc2 * (1.0 + 1e-5)); }

// whether a pair group's list holds a wide angular SF (kind 9): its triplets are not limited by r_jk
__device__ __forceinline__ bool group_has_wide(const AngularSF* list, int n) {
    bool w = false;
    for (int s = 0; s < n; ++s) w |= list[s].wide != 0;
    return w;
}

}  // namespace nnp

// stream.cuh -- triplet enumeration of the lane-owned design (k_sf / k_force fast paths).
//
// ncu of the first (queue) design showed both kernels bound by shared-memory bandwidth and
// instruction issue, not by the FP64 pipe (profiles/r1a_*): every triplet gathered both of its
// neighbours from shared memory, read-modify-wrote both force slots there, and 41 % of the
// instructions enumerated and compacted candidates.  Here a group of WPC warps (one CTA) owns one
// centre and shares its staged neighbourhood (more resident warps per byte of shared memory), and
//   * SCREENING is a lock-step loop in which lane l owns neighbour slot j = l (+32, ...) in
//     registers and tests it against its partners in FP32; the result is a BIT MASK per (pair
//     group, j) in shared memory -- no queue, no compaction traffic;
//   * the contributing triplets of ALL pair groups form one stream (group-major, then j, then
//     mask bit); a prefix sum of the mask popcounts splits it into NT EQUAL ranges, one per thread,
//     so every lane evaluates ceil(T/NT) triplets whatever the pass rate is;
//   * a lane walks its range bit by bit: j stays in registers until the mask of the next j starts
//     (data of j reloaded, j-side force sum flushed), only the partner k is gathered.
// Every mask word carries a 32-bit DESCRIPTOR (owner slot j, first partner slot, wrap bound and
// modulus), so that walking needs no group table: with 32 lanes on 32 different ranges, SOME lane
// moves to its next word or its next j in almost every iteration, and such a rare-per-lane step costs
// the whole warp its instructions (ncu r1b: ~100 of ~220 instructions per iteration of the first
// version were this bookkeeping).
// A pair group is either WITHIN one element segment (tournament: bit r-1 of slot j pairs it with
// slot (j + r) mod ns, r = 1..ns/2, each unordered pair once) or BETWEEN two segments (bit q of
// slot j of the first pairs it with slot q of the second).
#pragma once
#include "nnp_internal.h"

namespace nnp {

constexpr unsigned FULL = 0xffffffffu;

// one active pair group of the current centre; lives in per-CTA shared memory as three int4.
// Mask word (j, w) of the group sits at  woff + (j - jbeg) * stride + w.  Two stream orders:
//   group-major (k_sf):   a group's words are contiguous (stride = W) -> a lane changes group rarely;
//   j-major    (k_force): all words of slot j, over every group it owns, are contiguous
//                         (stride = sum of W over the groups of j's element) -> the lanes that share
//                         a slot j are consecutive, which makes the in-loop j-side flush conflict-free.
struct GroupTab {
    int jbeg, jend;   // slots owning masks: [jbeg, jend)
    int kbase;        // within: = jbeg; between: first slot of the partner segment
    int ns;           // within: segment size (wrap modulus); between: 0
    int W;            // mask words per j in this group
    int pair;         // pair-group index (coefficient tables, G positions)
    int woff;         // index of the mask word (jbeg, 0) of this group
    int nk;           // partners per j: within ns/2 rounds, between the partner segment's size
    int stride;       // words from (j, w) to (j + 1, w)
    int gfirst;       // first group of the block this group belongs to
    int last;         // 1 if this is the last group of its block
    int gmoff;        // index of this group's first word in GROUP-major order (the order of the exported masks)
};

// upper bound of the mask words of one centre with at most `cap` neighbours of `n_elem` elements:
// within: ns * ceil(floor(ns/2)/32) <= ns (ns/64 + 1); between: n1 * ceil(n2/32) <= n1 (n2/32 + 1);
// summed over the groups: <= n^2/64 + n * n_elem.  (The u16 prefix array of the kernels aliases a
// 16 B-per-slot region: 2 * (n^2/64 + 4 n) <= 16 * capacity holds for n <= 255.)
__host__ __device__ constexpr int mask_words_cap(int cap, int n_elem) { return cap * cap / 64 + cap * n_elem; }

// Builds the group table of the centre (uniform code; every thread computes the same, thread 0 stores).
// n_ang[pr] != 0 marks pair groups that have angular symmetry functions.  Returns #groups; NW out.
template <bool JMAJOR>
__device__ __forceinline__ int build_groups(const int* seg, int n_elem, const int32_t* n_ang, GroupTab* tab, int tid,
                                            int& NW) {
    int ng = 0, woff = 0, gm = 0;
    for (int e1 = 0; e1 < n_elem; ++e1) {
        const int n1 = seg[e1 + 1] - seg[e1];
        const int gfirst = ng;
        int wsum = 0;       // words per j over the groups of this block (j-major)
        for (int e2 = e1; e2 < n_elem; ++e2) {
            const int pr = pair_index(e1, e2, n_elem);
            if (n_ang[pr] == 0) continue;
            const int n2 = seg[e2 + 1] - seg[e2];
            GroupTab g;
            g.jbeg = seg[e1]; g.jend = seg[e1 + 1]; g.pair = pr;
            if (e1 == e2) { g.kbase = g.jbeg; g.ns = n1; g.nk = n1 / 2; }
            else { g.kbase = seg[e2]; g.ns = 0; g.nk = n1 > 0 ? n2 : 0; }
            g.W = (g.nk + 31) >> 5;
            if (g.W == 0) continue;
            g.gmoff = gm;
            gm += n1 * g.W;
            if (JMAJOR) { g.woff = woff + wsum; g.gfirst = gfirst; g.stride = 0; g.last = 0; wsum += g.W; }
            else { g.woff = woff; g.gfirst = ng; g.stride = g.W; g.last = 1; woff += n1 * g.W; }
            if (tid == 0) tab[ng] = g;
            ++ng;
        }
        if (JMAJOR && ng > gfirst) {
            if (tid == 0) {
                for (int t = gfirst; t < ng; ++t) tab[t].stride = wsum;
                tab[ng - 1].last = 1;
            }
            woff += n1 * wsum;
        }
    }
    NW = woff;
    return ng;
}

// number of mask words of a centre (= NW of build_groups, either order)
__device__ __forceinline__ int count_words(const int* seg, int n_elem, const int32_t* n_ang) {
    int nw = 0;
    for (int e1 = 0; e1 < n_elem; ++e1) {
        const int n1 = seg[e1 + 1] - seg[e1];
        for (int e2 = e1; e2 < n_elem; ++e2) {
            if (n_ang[pair_index(e1, e2, n_elem)] == 0) continue;
            const int nk = e1 == e2 ? n1 / 2 : (n1 > 0 ? seg[e2 + 1] - seg[e2] : 0);
            nw += n1 * ((nk + 31) >> 5);
        }
    }
    return nw;
}

// group-major word index y -> (group, local owner index, word)
__device__ __forceinline__ void decode_gmajor(const GroupTab* tab, int ng, int y, int& g, int& jl, int& w) {
    g = 0;
    for (int t = 1; t < ng; ++t)
        if (tab[t].gmoff <= y) g = t;
    const int rel = y - tab[g].gmoff, W = tab[g].W;
    jl = W == 1 ? rel : (W == 2 ? rel >> 1 : rel / W);
    w = rel - jl * W;
}

__device__ __forceinline__ bool close32(const float4 a, const float4 b, float rc2f) {
    const float wx = b.x - a.x, wy = b.y - a.y, wz = b.z - a.z;
    return fmaf(wx, wx, fmaf(wy, wy, wz * wz)) < rc2f;
}

// Descriptor of mask word w of owner slot j = jbeg + jl:
//     j | first << 8 | alt << 16 | bw << 24 | pair << 30
// Bit b of the word pairs j with slot  k = (b + (b < bw ? first : alt)) & 255:  `first` is the partner of
// bit 0, bw the first bit that wraps round the end of the segment (32 = none) and alt = segment start - bw
// (mod 256).  The pair-group index fits the two spare bits when there are at most two elements (three
// groups); with more elements the kernels derive it from the slots (pair_of_slots).
__device__ __forceinline__ uint32_t word_desc(const GroupTab& g, int jl, int w) {
    const uint32_t hi = (uint32_t)(g.pair & 3) << 30;
    if (g.ns > 0) {
        int kb = jl + 32 * w + 1;
        if (kb >= g.ns) kb -= g.ns;
        const int bw = min(g.ns - kb, 32);
        return (uint32_t)(g.jbeg + jl) | (uint32_t)(g.jbeg + kb) << 8 | (uint32_t)((g.jbeg - bw) & 255) << 16 |
               (uint32_t)bw << 24 | hi;
    }
    return (uint32_t)(g.jbeg + jl) | (uint32_t)(g.kbase + 32 * w) << 8 | 32u << 24 | hi;
}

// Screening of one group: FP32 test |u_k - u_j|^2 < rc^2 (1 + 1e-5) (never drops a contributing pair; the
// evaluation applies the exact FP64 test) -> words[woff + (j - jbeg) stride + w] = (mask, descriptor).
// Thread t owns slot j = jbeg + t (+nt, ...) in registers; within a group its partner walks (j + r) mod ns
// (distinct consecutive addresses), between groups all lanes test the same partner (broadcast load).
__device__ __forceinline__ void screen_group(const GroupTab g, const float4* f32, uint2* words, float rc2f, int tid,
                                             int nt) {
    const int nj = g.jend - g.jbeg;
    const int R = g.nk;
    for (int jb = tid & ~31; jb < nj; jb += nt) {        // warp-uniform trip count
        const int jl = jb + (tid & 31);
        const bool vj = jl < nj;
        const float4 a = f32[g.jbeg + (vj ? jl : 0)];
        uint2* dst = words + g.woff + jl * g.stride;
        uint32_t word = 0, bit = 1u;
        if (g.ns > 0) {
            // tournament inside the segment: round t pairs j with (j + t + 1) mod ns; with an even ns the
            // last round (t = R - 1) holds every pair twice -> only the lower half of the slots keeps it
            const int ns = g.ns;
            const float4* src = f32 + g.jbeg;
            int kl = vj ? jl : 0;
            const int Rfull = (ns & 1) ? R : R - 1;
            for (int t = 0; t < Rfull; ++t) {
                ++kl;
                if (kl >= ns) kl -= ns;
                if (close32(a, src[kl], rc2f)) word |= bit;
                bit <<= 1;
                if ((t & 31) == 31) {
                    if (vj) dst[t >> 5] = make_uint2(word, word_desc(g, jl, t >> 5));
                    word = 0; bit = 1u;
                }
            }
            if (Rfull < R) {
                ++kl;
                if (kl >= ns) kl -= ns;
                if (jl < R && close32(a, src[kl], rc2f)) word |= bit;
            }
            if (vj && ((R & 31) != 0 || Rfull < R)) dst[(R - 1) >> 5] = make_uint2(word, word_desc(g, jl, (R - 1) >> 5));
        } else {
            const float4* src = f32 + g.kbase;
            for (int t = 0; t < R; ++t) {
                if (close32(a, src[t], rc2f)) word |= bit;       // uniform address: broadcast
                bit <<= 1;
                if ((t & 31) == 31) {
                    if (vj) dst[t >> 5] = make_uint2(word, word_desc(g, jl, t >> 5));
                    word = 0; bit = 1u;
                }
            }
            if (vj && (R & 31) != 0) dst[(R - 1) >> 5] = make_uint2(word, word_desc(g, jl, (R - 1) >> 5));
        }
    }
}

// Exclusive prefix of the mask popcounts -> C[0..NW) (u16; T <= 255*254/2 fits); returns T.
// Block-wide: nt = 32 * nwarp threads; wsum = nwarp ints of shared scratch.  Contains __syncthreads.
__device__ __forceinline__ int mask_prefix(const uint2* words, uint16_t* C, int NW, int tid, int nt, int* wsum) {
    const int lane = tid & 31, wid = tid >> 5, nwarp = nt >> 5;
    const int chunk = (NW + nt - 1) / nt;
    const int beg = min(tid * chunk, NW), end = min(beg + chunk, NW);
    int s = 0;
    for (int x = beg; x < end; ++x) s += __popc(words[x].x);
    int incl = s;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int t = __shfl_up_sync(FULL, incl, d);
        if (lane >= d) incl += t;
    }
    if (lane == 31) wsum[wid] = incl;
    __syncthreads();
    int base = 0, total = 0;
    for (int w = 0; w < nwarp; ++w) {
        const int v = wsum[w];
        if (w < wid) base += v;
        total += v;
    }
    int run = base + incl - s;
    for (int x = beg; x < end; ++x) {
        C[x] = (uint16_t)run;
        run += __popc(words[x].x);
    }
    return total;
}

// A lane's position in the triplet stream.
struct Walker {
    const uint2* words;
    int idx;          // current word
    uint32_t m;       // bits of the current word not yet visited (kept non-zero once the lane is done)
    uint32_t d;       // descriptor of the current word
    int cnt;          // triplets left for this lane

    __device__ __forceinline__ int j() const { return (int)(d & 255u); }
    __device__ __forceinline__ int first_partner() const { return (int)((d >> 8) & 255u); }
    __device__ __forceinline__ int pair2() const { return (int)(d >> 30); }     // valid when n_elem <= 2

    // position the lane at triplet number S of the stream (cnt > 0 required)
    __device__ __forceinline__ void seek(const uint16_t* C, int NW, int S) {
        int lo = 0, hi = NW - 1;                   // largest idx with C[idx] <= S
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if ((int)C[mid] <= S) lo = mid; else hi = mid - 1;
        }
        idx = lo;
        const uint2 w = words[idx];
        m = w.x;
        d = w.y;
        for (int s = S - (int)C[idx]; s > 0; --s) m &= m - 1;
    }

    // move the lane to its next non-empty word if it has run out of bits (plain divergent loop)
    __device__ __forceinline__ void advance() {
        while (m == 0u) {
            ++idx;
            const uint2 w = words[idx];
            m = w.x;
            d = w.y;
        }
    }

    // pop the next triplet of the lane: partner slot k
    __device__ __forceinline__ int pop() {
        const int b = __ffs(m) - 1;
        m &= m - 1;
        if (--cnt == 0) m = 1u;                    // done: never advance past the lane's range
        const uint32_t sel = b < (int)((d >> 24) & 63u) ? d >> 8 : d >> 16;
        return (int)((sel + (uint32_t)b) & 255u);
    }
};

// pair-group index of (owner slot j, partner slot k) from the segment boundaries (element of j <= element of k)
__device__ __forceinline__ int pair_of_slots(int j, int k, const int* seg, int n_elem) {
    const int ej = (j >= seg[1]) + (j >= seg[2]) + (j >= seg[3]);
    const int ek = (k >= seg[1]) + (k >= seg[2]) + (k >= seg[3]);
    return pair_index(ej, ek, n_elem);
}

}  // namespace nnp

// k_sf2.cu -- S2 fast path (specialised pair groups): atom-centred symmetry functions G_i, radial
// G2 and angular G3 (PAPER.md L40 step 1; formulas: include/nnp.h at nnp_sf, readings 2-4).
// Lane-owned design (stream.cuh), same staging / screening / stream split as k_force2.cu: one CTA of
// WPC warps per centre; a lane keeps neighbour j in registers and gathers only the partner k.  The
// stream is GROUP-major here, so a lane changes pair group at most (#groups - 1) times per centre: it
// accumulates the NACC values of its current group in registers and hands them over (shared-memory
// atomics, rare) when its group changes; at the end the lanes of a warp are reduced per group.
#include "angular.cuh"
#include "geometry.cuh"
#include "stream.cuh"

namespace nnp {

struct Sf2Params {
    int64_t n;
    int n_elem, ncell, stride, cap, g_stride;
    int pass;                            // free-eta kernels: which AngPass of the element's program this launch evaluates
    double rc, rc2, k2;                  // k2 = (pi / (2 rc))^2
    double box[3], half[3];
    const double *sx, *sy, *sz;
    const int32_t *cell_start, *nbr, *nbr_cnt;
    double* G;
    const int64_t* word_off;             // mask export (see Workspace::gmask)
    uint32_t* gmask;
    int64_t gmask_cap;
    const ElemProgram* prog[MAX_ELEM];
    int variant[MAX_ELEM];
};

// Shared memory of one centre: planes p0 (ux,uy), p1 (uz,1/a), p2 (exp(-eta0 a^2), fc(a)) double2[CAPA];
// ra (a) double[CAPA]; FP32 screening copy float4[CAPA] (the prefix array aliases it afterwards);
// then group table, G accumulators [npair][NACC], scratch, mask words (mask + descriptor)
// arithmetic type R of the staged planes and the per-triplet evaluation (double, or float in the opt-in
// mixed-precision mode: see k_force2.cu)
template <class R> struct SfVec2;
template <> struct SfVec2<double> { using type = double2; };
template <> struct SfVec2<float> { using type = float2; };
__device__ __forceinline__ double2 sf_mk2(double a, double b) { return make_double2(a, b); }
__device__ __forceinline__ float2 sf_mk2(float a, float b) { return make_float2(a, b); }

template <class Spec>
__host__ __device__ constexpr size_t sf2_smem(int capa, int n_elem, int wpc, size_t real = 8) {
    const size_t npair = (size_t)n_elem * (n_elem + 1) / 2;
    size_t b = (size_t)capa * (3 * 2 * real + 8 + 16);
    b += npair * sizeof(GroupTab);
    b += (size_t)(wpc + 1) * npair * Spec::NACC * 8;
    b += 64;
    b += (size_t)mask_words_cap(capa, n_elem) * 8;
    return (b + 15) / 16 * 16;
}

#ifndef S2_MINB1
#define S2_MINB1 24          // resident CTAs per SM asked of the one-warp-per-centre instantiation (12 SFs per group)
#endif
#ifndef S2_MINB_F32
#define S2_MINB_F32 32       // warps per SM asked of the FP32 instantiations (mixed-precision mode)
#endif
template <class Spec, int WPC, int CAPA, bool TINY, class R>
__global__ void __launch_bounds__(WPC * 32, WPC == 1 ? (Spec::NACC <= 12 ? S2_MINB1 : 16) : (sizeof(R) == 4 ? (Spec::NACC <= 12 ? S2_MINB_F32 : 20) : (Spec::NACC <= 12 ? 24 : (Spec::NACC <= 16 ? 20 : 16))) / WPC) k_sf2(const __grid_constant__ Sf2Params p) {
    using R2 = typename SfVec2<R>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NT = WPC * 32;
    constexpr int NACC = Spec::NACC;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int64_t i = blockIdx.x;
    int tc = 0;
    for (int e = 1; e < p.n_elem; ++e)
        if (i >= p.cell_start[(size_t)e * p.ncell]) tc = e;
    if (p.variant[tc] != Spec::ID && !(Spec::FREE_ETA && p.variant[tc] == ANG_MULTI)) return;          // uniform per CTA
    const ElemProgram* __restrict__ prog = p.prog[tc];
    // free-eta kernels: one launch per pass (nnp_internal.h AngPass); BASELINE.json's shapes: one sweep at the global rc
    const AngPass* __restrict__ ps = &prog->pass[Spec::FREE_ETA ? p.pass : 0];
    if (Spec::FREE_ETA && (p.pass >= prog->n_pass || ps->spec != Spec::ID)) return;
    const bool own_rc = Spec::FREE_ETA && ps->own_rc != 0;          // the pass's cutoff is shorter than the neighbour list's
    const bool widep = Spec::FREE_ETA && ps->wide != 0;             // wide angular functions: no r_jk term, every pair counts
    const int z0 = Spec::FREE_ETA ? ps->zeta0 : 1;                  // menu bits 0, 1, 2 stand for zeta = z0, 2 z0, 4 z0 ...
    const int zx = Spec::FREE_ETA ? ps->zeta_x : 16;                // ... and bit 4 for zeta = zx (16 z0: two more squarings)
    const bool zx_own = Spec::FREE_ETA && zx != 16 * z0;
    const double rc2p = Spec::FREE_ETA ? ps->rc2 : p.rc2, k2p = Spec::FREE_ETA ? ps->k2 : p.k2;
    const int32_t* __restrict__ n_ang = Spec::FREE_ETA ? ps->n_ang : prog->n_ang;
    const bool first_pass = !Spec::FREE_ETA || p.pass == 0;         // the radial block and the tail of the G row
    const bool handover = !Spec::FREE_ETA || (prog->n_pass == 1 && !own_rc && !widep);   // masks to the force kernel

    constexpr int capa = CAPA;
    const int npair = p.n_elem * (p.n_elem + 1) / 2;
    R2* p0 = reinterpret_cast<R2*>(smem_raw);               // (ux, uy)
    R2* p1 = p0 + capa;                                     // (uz, 1/a)
    R2* p2 = p1 + capa;                                     // (exp(-eta_0 a^2), fc(a))
    double* ra = reinterpret_cast<double*>(p2 + capa);      // a (FP64 in both modes: the radial block)
    float4* f32 = reinterpret_cast<float4*>(ra + capa);     // screening copy
    uint16_t* C = reinterpret_cast<uint16_t*>(f32);         // alias: prefix of the mask popcounts (after screening)
    GroupTab* tab = reinterpret_cast<GroupTab*>(f32 + capa);
    // [WPC + 1][pair][NACC]: set 0 = sums handed over by the one lane that leaves a group inside its range,
    // set 1 + w = sums of the lanes of warp w that end in the group; added in this fixed order (the energies
    // must not depend on scheduling)
    double* gacc = reinterpret_cast<double*>(tab + npair);
    int* wsum = reinterpret_cast<int*>(gacc + (WPC + 1) * npair * NACC);
    uint2* words = reinterpret_cast<uint2*>(wsum + 16);     // (mask, descriptor)

    int seg[MAX_ELEM + 1];
    seg[0] = 0;
#pragma unroll
    for (int e = 0; e < MAX_ELEM; ++e) seg[e + 1] = seg[e] + p.nbr_cnt[(size_t)i * MAX_ELEM + e];
    const int ntot = seg[MAX_ELEM];

    // ---- stage the neighbourhood -------------------------------------------------------------------
    const double xi = p.sx[i], yi = p.sy[i], zi = p.sz[i];
    const int32_t* row = p.nbr + (size_t)i * p.stride;
    const double eta0 = prog->ang_eta[0];
    const int neta = Spec::FREE_ETA ? ps->n_eta : Spec::NETA;
    R etav[Spec::FREE_ETA ? Spec::NETA : 1];
    if constexpr (Spec::FREE_ETA)
        for (int e = 0; e < Spec::NETA; ++e) etav[e] = (R)ps->eta[e];
    const R eta0r = (R)eta0, k2r = (R)k2p, rc2r = (R)rc2p;
    constexpr bool tiny = TINY;                      // exp(-eta_0 r^2) without range reduction (mathfn.cuh exp_tiny)
    if ((prog->tiny_exp != 0) != TINY) return;       // uniform per CTA: the other instantiation owns this element
    for (int m = tid; m < ntot; m += NT) {
        const int j = row[m];
        const double dx = min_image_1d(xi, p.sx[j], p.box[0], p.half[0]);
        const double dy = min_image_1d(yi, p.sy[j], p.box[1], p.half[1]);
        const double dz = min_image_1d(zi, p.sz[j], p.box[2], p.half[2]);
        const double a2 = fma(dx, dx, fma(dy, dy, dz * dz));
        const double ia = rsqrt(a2);
        const bool in = !own_rc || a2 < rc2p;                // beyond the pass's radius: fc = 0, and out of the screening
        const double Ca = in ? cos_only(a2 * k2p) : 0.0;
        p0[m] = sf_mk2((R)dx, (R)dy);
        p1[m] = sf_mk2((R)dz, (R)ia);
        // first component: exp(-eta_0 a^2), or a^2 itself where every eta gets its own exponential (FREE_ETA)
        p2[m] = sf_mk2((R)(Spec::FREE_ETA ? a2 : (tiny ? exp_tiny(-eta0 * a2) : exp_small(-eta0 * a2))), (R)(Ca * Ca));
        ra[m] = a2 * ia;
        f32[m] = in ? make_float4((float)dx, (float)dy, (float)dz, 0.f) : make_float4(1e9f * (float)(m + 1), 0.f, 0.f, 0.f);
    }
    for (int s = tid; s < (WPC + 1) * npair * NACC; s += NT) gacc[s] = 0.0;
    int NW = 0;
    const int ng = build_groups<false>(seg, p.n_elem, n_ang, tab, tid, NW);
    __syncthreads();

    double* Grow = p.G + (size_t)i * p.g_stride;
    if (first_pass)
        for (int s = prog->n_sf + tid; s < p.g_stride; s += NT) Grow[s] = 0.0;

    // ---- radial: G = sum_j exp(-eta (a - rs)^2) fc(a) over the neighbours of element e; one warp per SF
    // (first pass only; with cutoff radii per symmetry function the generic kernel's radial-only mode does it, k_sf.cu)
    for (int e = 0; e < ((first_pass && prog->per_sf_rc == 0) ? p.n_elem : 0); ++e) {
        const int nr = prog->n_rad[e], off = prog->rad_off[e];
        for (int r = wid; r < nr; r += WPC) {
            const RadialSF f = prog->rad[off + r];
            double acc = 0.0;
            for (int m = seg[e] + lane; m < seg[e + 1]; m += 32) {
                const double d = ra[m] - f.rs;
                acc = fma(exp_small(fmax(-f.eta * d * d, -700.0)), (double)p2[m].y, acc);
            }
            acc = warp_sum(acc);
            if (lane == 0) Grow[f.g] = acc;
        }
    }

    // ---- screening -> masks; prefix; even split of the triplet stream over the NT threads ------------
    const float rc2f = widep ? 3.0e38f : (float)(rc2p * (1.0 + 1e-5));      // wide: no screening (a switched-off slot has fc = 0)
    for (int g = 0; g < ng; ++g) screen_group(tab[g], f32, words, rc2f, tid, NT);
    __syncthreads();
    // hand the masks to the force kernel (this kernel's group-major order), if they fit the budget
    {
        const int64_t off = p.word_off[i];
        if (handover && off + NW <= p.gmask_cap)
            for (int x = tid; x < NW; x += NT) p.gmask[off + x] = words[x].x;
    }
    const int T = mask_prefix(words, C, NW, tid, NT, wsum);
    __syncthreads();
    const int quota = (T + NT - 1) / NT;
    Walker wk;
    wk.words = words;
    wk.cnt = max(0, min(quota, T - tid * quota));
    wk.m = 1u; wk.d = 0u; wk.idx = 0;
    if (wk.cnt > 0) wk.seek(C, NW, tid * quota);

    // ---- angular part: every lane walks its range of the stream ---------------------------------------
    R jx = (R)1, jy = (R)1, jz = (R)1, jia = (R)1, je0 = (R)1, jfa = (R)0;
    int jcur = -1, paircur = -1;
    uint32_t dcur = 0xffffffffu;
    R acc[NACC];                                     // FP32 mode: a lane sums its ~30 triplets in FP32, the lanes are reduced in FP64
#pragma unroll
    for (int a = 0; a < NACC; ++a) acc[a] = (R)0;
    for (int it = 0; it < quota; ++it) {
        const bool active = wk.cnt > 0;
        wk.advance();
        if (active && wk.d != dcur) {
            dcur = wk.d;
            const int jn = wk.j();
            if (jn != jcur) {
                jcur = jn;
                const R2 a0 = p0[jcur], a1 = p1[jcur], a2 = p2[jcur];
                jx = a0.x; jy = a0.y; jz = a1.x; jia = a1.y; je0 = a2.x; jfa = a2.y;
            }
            const int pr = p.n_elem <= 2 ? wk.pair2() : pair_of_slots(jn, wk.first_partner(), seg, p.n_elem);
            if (pr != paircur) {
                // The lane enters another pair group: hand the sums over.  Only ONE lane of the CTA leaves a
                // given group inside its range (the group-major stream is split into contiguous ranges),
                // so this is a plain store.
                if (paircur >= 0) {
#pragma unroll
                    for (int a = 0; a < NACC; ++a) {
                        gacc[paircur * NACC + a] = (double)acc[a];
                        acc[a] = (R)0;
                    }
                }
                paircur = pr;
            }
        }
        const int k = active ? wk.pop() : max(jcur, 0);
        const R2 k0 = p0[k], k1 = p1[k], k2v = p2[k];
        const R wx = k0.x - jx, wy = k0.y - jy, wz = k1.x - jz;
        const R c2 = fma(wx, wx, fma(wy, wy, wz * wz));
        const R Cc = cos_only(c2 * k2r);
        R Cf = (jfa * k2v.y) * (Cc * Cc);           // fc(a) fc(b) fc(c), fc(c) = cos^2(pi c / (2 rc))
        if (widep) Cf = jfa * k2v.y;                // wide: fc(a) fc(b) only
        if (!active || (!widep && !(c2 < rc2r))) Cf = (R)0;     // cutoff (FP64: exact; the masks were screened in FP32)
        R Y[Spec::NETA];
        const R r2 = widep ? je0 + k2v.x : (je0 + k2v.x) + c2;   // FREE_ETA: a^2 + b^2 (+ c^2, narrow) -- the staged value is a^2
        if constexpr (!Spec::FREE_ETA) {
            Y[0] = (je0 * k2v.x) * (tiny ? exp_tiny5(-eta0r * c2) : exp_small(-eta0r * c2));   // degree 5: 1e-14 (46.9 -> 46.7 ms)
            if constexpr (Spec::NETA > 1) Y[1] = ipow<Spec::ratio(1)>(Y[Spec::rbase(1)]);
            if constexpr (Spec::NETA > 2) Y[2] = ipow<Spec::ratio(2)>(Y[Spec::rbase(2)]);
            if constexpr (Spec::NETA > 3) Y[3] = ipow<Spec::ratio(3)>(Y[Spec::rbase(3)]);
        }
        const R cosv = fma(jx, k0.x, fma(jy, k0.y, jz * k1.x)) * (jia * k1.y);
        R pw[2][Spec::MAXBIT + 1];
        pw[0][0] = (R)1 + cosv;
        pw[1][0] = (R)1 - cosv;
        const R base0 = pw[0][0], base1 = pw[1][0];
        if (Spec::FREE_ETA && z0 > 1) {                        // uniform per CTA
            pw[0][0] = powi_uniform(pw[0][0], z0);
            pw[1][0] = powi_uniform(pw[1][0], z0);
        }
#pragma unroll
        for (int b = 1; b <= Spec::MAXBIT; ++b) {
            pw[0][b] = pw[0][b - 1] * pw[0][b - 1];
            pw[1][b] = pw[1][b - 1] * pw[1][b - 1];
        }
        if (zx_own) {                                          // uniform per CTA: the top menu entry is an exponent of its own
            pw[0][Spec::MAXBIT] = powi_uniform(base0, zx);
            pw[1][Spec::MAXBIT] = powi_uniform(base1, zx);
        }
#pragma unroll
        for (int e = 0; e < Spec::NETA; ++e) {
            if (Spec::FREE_ETA && e >= neta) break;            // uniform per CTA: eta slots the table does not use
            if constexpr (Spec::FREE_ETA) Y[e] = exp_small(-etav[e] * r2);
            const R xc = Y[e] * Cf;
#pragma unroll
            for (int b = 0; b <= Spec::MAXBIT; ++b) {
                if (Spec::mask(e) >> b & 1u) acc[acc_index<Spec>(e, b)] = fma(pw[0][b], xc, acc[acc_index<Spec>(e, b)]);
                if (Spec::mask(e) >> (8 + b) & 1u)
                    acc[acc_index<Spec>(e, 8 + b)] = fma(pw[1][b], xc, acc[acc_index<Spec>(e, 8 + b)]);
            }
        }
    }
    // ---- reduce: per pair group present in the warp, sum the lanes that ended in it -------------------
    constexpr int NR = NACC <= 16 ? 16 : 32;
    for (int pr = 0; pr < npair; ++pr) {
        if (!__any_sync(FULL, paircur == pr)) continue;
        double v[NR];
#pragma unroll
        for (int a = 0; a < NR; ++a) v[a] = (a < NACC && paircur == pr) ? (double)acc[a < NACC ? a : 0] : 0.0;
        warp_reduce_multi<NR>(v, lane);
        const int a = warp_reduce_index<NR>(lane);
        if ((lane & (32 / NR - 1)) == 0 && a < NACC) gacc[((1 + wid) * npair + pr) * NACC + a] = v[0];
    }
    __syncthreads();
    // ---- G = 2^(1-zeta) * sum ---------------------------------------------------------------------------
    for (int s = tid; s < npair * 16 * Spec::NETA; s += NT) {
        const int pr = s / (16 * Spec::NETA), rem = s - pr * 16 * Spec::NETA;
        const int e = rem >> 4, b = rem & 15;
        bool on = false;
        int a = 0;
#pragma unroll
        for (int ee = 0; ee < Spec::NETA; ++ee) {
            const unsigned mk = Spec::mask(ee);
            if (ee < e) a += __popc(mk);
            else if (ee == e) { a += __popc(mk & ((1u << b) - 1u)); on = (mk >> b) & 1u; }
        }
        if (!on || n_ang[pr] == 0) continue;
        const int g = Spec::FREE_ETA ? ps->g[pr][e][b] : prog->ang_g[pr][e][b];
        if (g >= 0) {
            double tot = gacc[pr * NACC + a];
#pragma unroll
            for (int w = 0; w < WPC; ++w) tot += gacc[((1 + w) * npair + pr) * NACC + a];
            Grow[g] = exp2((double)(1 - ((b & 7) == Spec::MAXBIT ? zx : z0 << (b & 7)))) * tot;
        }
    }
}

// ---- mask words per centre and their prefix -----------------------------------------------------------
__global__ void __launch_bounds__(256)
k_count_words(int64_t n, int n_elem, int ncell, const int32_t* __restrict__ cell_start,
              const int32_t* __restrict__ nbr_cnt, const ElemProgram* p0, const ElemProgram* p1, const ElemProgram* p2,
              const ElemProgram* p3, int32_t* __restrict__ nw, int32_t* __restrict__ big_list, int32_t* __restrict__ big_count) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int tc = 0;
    for (int e = 1; e < n_elem; ++e)
        if (i >= cell_start[(size_t)e * ncell]) tc = e;
    const ElemProgram* prog = tc == 0 ? p0 : (tc == 1 ? p1 : (tc == 2 ? p2 : p3));
    int seg[MAX_ELEM + 1];
    seg[0] = 0;
#pragma unroll
    for (int e = 0; e < MAX_ELEM; ++e) seg[e + 1] = seg[e] + nbr_cnt[(size_t)i * MAX_ELEM + e];
    nw[i] = count_words(seg, n_elem, prog->n_ang);
    // centres that do not fit the 128-slot force kernel (k_force2.cu launch_one2); any order
    if (seg[MAX_ELEM] > 128) big_list[atomicAdd(big_count, 1)] = (int32_t)i;
}

int launch_word_offsets(const Workspace& w, const Grid& g, int64_t n, int n_elem, const ElemProgram* const* d_prog,
                        cudaStream_t st) {
    if (n == 0) return 0;
    const ElemProgram* pr[MAX_ELEM];
    for (int e = 0; e < MAX_ELEM; ++e) pr[e] = e < n_elem ? d_prog[e] : nullptr;
    k_count_words<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, n_elem, g.ncell, w.cell_start, w.nbr_cnt, pr[0], pr[1],
                                                                pr[2], pr[3], w.nw, w.big_list, w.status + 2);
    return 1 + launch_scan_i64_from_i32(w.nw, n, w.word_off, w.word_tmp, st);
}

#ifndef NNP_SF2_WPC
#define NNP_SF2_WPC 2
#endif
constexpr int SF2_WPC = NNP_SF2_WPC;

template <class Spec, int CAPA, bool TINY, class R, int WPC = SF2_WPC>
static int launch_capa_sf(const Sf2Params& p, cudaStream_t st) {
    const size_t smem = sf2_smem<Spec>(CAPA, p.n_elem, WPC, sizeof(R));
    static unsigned long long configured = 0ull;      // per device (opt_in_smem)
    opt_in_smem(k_sf2<Spec, WPC, CAPA, TINY, R>, &configured);
    k_sf2<Spec, WPC, CAPA, TINY, R><<<(unsigned)p.n, WPC * 32, smem, st>>>(p);
    return 1;
}

template <class Spec, bool TINY, class R = double>
static int launch_one_sf2(const Sf2Params& p, cudaStream_t st) {
    // small neighbourhoods (metals: ~20 neighbours, ~60 triplets per centre): 64 slots, ONE warp per centre
    if (p.cap <= 64) return launch_capa_sf<Spec, 64, TINY, double, 1>(p, st);
    // one launch at the slot capacity of max_neighbors (a 128 / 160 split as in k_force2.cu bought nothing here:
    // 48.19 vs 48.20 ms on configs[3] at 12 and 14 CTAs per SM -- this kernel is issue-bound, not occupancy-bound)
    if (p.cap <= 128) return launch_capa_sf<Spec, 128, TINY, R>(p, st);
    if (p.cap <= 160) return launch_capa_sf<Spec, 160, TINY, R>(p, st);
    return launch_capa_sf<Spec, 256, TINY, double>(p, st);
}

// launches the fast kernels for the specialised variants in use
int launch_sf2(const Workspace& w, const Grid& g, int64_t n, int n_elem, const ElemProgram* const* d_prog,
               const int* variant, const PassInfo& passes, double rc, int stride, int max_nbr, int g_stride, int precision,
               cudaStream_t st) {
    if (n == 0) return 0;
    Sf2Params p;
    p.n = n; p.n_elem = n_elem; p.ncell = g.ncell; p.stride = stride; p.cap = max_nbr; p.g_stride = g_stride; p.pass = 0;
    p.rc = rc; p.rc2 = rc * rc;
    p.k2 = (3.14159265358979323846 / (2.0 * rc)) * (3.14159265358979323846 / (2.0 * rc));
    for (int c = 0; c < 3; ++c) { p.box[c] = g.box[c]; p.half[c] = g.half[c]; }
    p.sx = w.sx; p.sy = w.sy; p.sz = w.sz;
    p.cell_start = w.cell_start; p.nbr = w.nbr; p.nbr_cnt = w.nbr_cnt; p.G = w.G;
    p.word_off = w.word_off; p.gmask = w.gmask; p.gmask_cap = w.gmask_cap;
    bool use[ANG_NVARIANT][2] = {};                                       // [variant][tiny_exp]
    for (int e = 0; e < MAX_ELEM; ++e) {
        p.prog[e] = e < n_elem ? d_prog[e] : nullptr;
        p.variant[e] = e < n_elem ? (variant[e] & 255) : -1;                 // bit 8 of variant[] = tiny_exp of the element
        if (e < n_elem) use[variant[e] & 255][(variant[e] >> 8) & 1] = true;
    }
    int launches = 0;
    const bool f32 = precision == 1;     // nnp_set_precision: mixed (BASELINE.json's two shapes only)
    if (max_nbr <= 32) {     // small neighbourhoods (metals): 8 lanes per centre (k_small.cu)
        if (use[ANG_BASE12][1]) launches += launch_sf_small(w, g, n, n_elem, d_prog, variant, rc, stride, max_nbr, g_stride, true, st);
        if (use[ANG_BASE12][0]) launches += launch_sf_small(w, g, n, n_elem, d_prog, variant, rc, stride, max_nbr, g_stride, false, st);
        use[ANG_BASE12][0] = use[ANG_BASE12][1] = false;
    }
    if (use[ANG_BASE12][1]) launches += f32 ? launch_one_sf2<SpecBase12, true, float>(p, st) : launch_one_sf2<SpecBase12, true>(p, st);
    if (use[ANG_BASE12][0]) launches += launch_one_sf2<SpecBase12, false>(p, st);
    if (use[ANG_WIDE32][1]) launches += f32 ? launch_one_sf2<SpecWide32, true, float>(p, st) : launch_one_sf2<SpecWide32, true>(p, st);
    if (use[ANG_WIDE32][0]) launches += launch_one_sf2<SpecWide32, false>(p, st);
    // free-eta tables: one launch per pass and kernel (the CTAs of elements without that pass return at once)
    for (int q = 0; q < MAX_PASS; ++q) {
        bool f32p = false, f16p = false;
        for (int e = 0; e < n_elem; ++e)
            if (q < passes.n_pass[e]) { f32p |= passes.spec[e][q] == ANG_FREE32; f16p |= passes.spec[e][q] == ANG_FREE16; }
        p.pass = q;
        if (f32p) launches += launch_one_sf2<SpecFree32, false>(p, st);
        if (f16p) launches += launch_one_sf2<SpecFree16, false>(p, st);
    }
    return launches;
}

}  // namespace nnp

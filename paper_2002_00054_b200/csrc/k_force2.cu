// k_force2.cu -- S4 fast path (specialised pair groups): forces F_m = - sum_i sum_s beta_is dG_is/dr_m
// with dG/dr RECOMPUTED, never stored (PAPER.md L40 step 3, L56-58, L98, L124); "the dominant
// angular force loop" (L116).  Lane-owned design (stream.cuh): one CTA of WPC warps per centre i; the
// centre's contributing triplets (i; j,k) are split evenly over the threads; a lane keeps neighbour j
// in registers, gathers only the partner k, accumulates the force on j in registers and the force on
// k in its warp's per-slot shared-memory accumulator (lanes of a warp that hit the same slot take
// turns; the turn order comes from match.any, issued early so that its latency hides).
//
// Per triplet, with u = r_j - r_i, v = r_k - r_i, w = v - u, the beta-weighted gradient is
//     dg/du = f_uu u + f_uv v - f_w w,      dg/dv = f_vv v + f_uv u + f_w w
// so  F_j = -s1 u + s3 v,  F_k = -s2 v + s3 u  with s1 = f_uu + f_w, s2 = f_vv + f_w, s3 = f_w - f_uv.
// The force on j is kept as (A = sum s1, V = sum s3 v) in registers while the lane owns j and folded
// into the slot accumulator as V - A u when the lane leaves j; the force on k goes straight into the
// slot accumulator (three doubles per slot).  F_slot - R u (R = radial part) is flushed with one global
// FP64 RED per component per neighbour; the centre receives minus the sum.
//
// Coefficients: the lane keeps c_b = beta_b 2^(1-zeta_b) of its current pair group in registers
// (NACC <= 12; larger sets load them per eta as 128-bit pairs) -- per-lane table loads from shared memory
// cost 4 wavefronts each (ncu, r1b) -- and gets
// dP/dcos from the SAME coefficients with pre-scaled powers zeta (1 +- cos)^(zeta-1): the factor zeta =
// 2^b is an integer add on the exponent field, the factor lambda a negated operand.
#include "angular.cuh"
#include "geometry.cuh"
#include "stream.cuh"

namespace nnp {

struct Force2Params {
    int64_t n;
    int n_elem, ncell, stride, cap, g_stride;
    int nt_lo, nt_hi;                    // this launch owns the centres with nt_lo <= neighbours <= nt_hi (slot-capacity split)
    int pass;                            // free-eta kernels: which AngPass of the element's program this launch evaluates
    double rc, rc2, k2;                  // k2 = (pi / (2 rc))^2
    double box[3], half[3];
    const double *sx, *sy, *sz;
    const int32_t *cell_start, *nbr, *nbr_cnt;
    const double* dEdG;
    double* f_sorted;
    int fixed;                           // 1: fixed-point force accumulation (nnp_internal.h force_add)
    int32_t *status, *sticky;
    const int32_t *big_list, *big_count; // centres with more than 128 neighbours (k_count_words)
    const int64_t* word_off;             // masks from the SF kernel (see Workspace::gmask)
    const uint32_t* gmask;
    int64_t gmask_cap;
    const ElemProgram* prog[MAX_ELEM];
    int variant[MAX_ELEM];
};

template <class Spec>
__host__ __device__ constexpr int bt2_stride() { return Spec::NACC + 1; }   // +1: groups land on different banks

// Shared memory of one centre (= one CTA of WPC warps).  CAPA (slot capacity) is a template parameter so
// that every array of the hot loop sits at a compile-time offset (ncu r1b: with run-time plane offsets
// the loop spent ~40 of its ~380 instructions re-deriving shared-memory addresses):
//   planes p0,p1,p2 (double2[CAPA]) | WPC accumulator sets: fxy double2[CAPA], fz double[CAPA], 8 B pad
//   (the FP32 screening copy and the prefix array alias set 0) | e0, rad double[CAPA] |
//   then, at run-time offsets: group table, coefficient tables, scratch, beta row, and the mask words
//   (mask + descriptor, uint2[mask_words_cap(CAPA, n_elem)])
template <class Spec>
__host__ __device__ constexpr size_t force2_smem(int capa, int g_stride, int n_elem, int wpc, size_t real = 8) {
    const size_t npair = (size_t)n_elem * (n_elem + 1) / 2;
    size_t b = (size_t)capa * (3 * 2 * real + 2 * real + (size_t)wpc * 4 * real) + 8;
    b += npair * sizeof(GroupTab);
    b += npair * bt2_stride<Spec>() * 2 * real;
    b += 64 + (size_t)((g_stride + 1) & ~1) * 8;
    b += (size_t)mask_words_cap(capa, n_elem) * 8;
    return (b + 15) / 16 * 16;
}

// Arithmetic type of the staged planes, the per-triplet evaluation and the per-slot accumulators: double (the
// default, BASELINE.json's FP64) or float (nnp_set_precision(NNP_PRECISION_MIXED): FP32 staging and
// triplet arithmetic, FP64 staging geometry, radial part, networks and global force / energy accumulation).
template <class R> struct Vec2;
template <> struct Vec2<double> { using type = double2; };
template <> struct Vec2<float> { using type = float2; };
__device__ __forceinline__ double2 mk2(double a, double b) { return make_double2(a, b); }
__device__ __forceinline__ float2 mk2(float a, float b) { return make_float2(a, b); }

template <class R>
struct SlotAcc2 {
    typename Vec2<R>::type* fxy;  // (Fx, Fy)
    R* fz;                        // Fz
};

// rank of the lane among the lanes of its warp that target the same slot (inactive lanes: 0)
__device__ __forceinline__ int conflict_rank(int slot, bool act, int lane) {
    const unsigned peers = __match_any_sync(FULL, act ? slot : -1 - lane);
    return __popc(peers & ((1u << lane) - 1u));
}

// acc[slot] += (x, y, z) for the lanes with act; lanes that target the same slot take turns
template <class R>
__device__ __forceinline__ void slot_add(const SlotAcc2<R>& acc, int slot, bool act, int rank, R x, R y, R z) {
    for (int pass = 0; __any_sync(FULL, act && rank >= pass); ++pass) {
        if (act && rank == pass) {
            typename Vec2<R>::type p = acc.fxy[slot];
            R q = acc.fz[slot];
            p.x += x; p.y += y; q += z;
            acc.fxy[slot] = p;
            acc.fz[slot] = q;
        }
        __syncwarp();
    }
}

// x * 2^b for b >= 0 by an integer add on the exponent field (x >= 0 finite, far from overflow; x = 0
// becomes 2^(b-1023), which is harmless where it is used)
__device__ __forceinline__ double scale2(double x, int b) {
    return __hiloint2double(__double2hiint(x) + (b << 20), __double2loint(x));
}
__device__ __forceinline__ float scale2(float x, int b) { return __int_as_float(__float_as_int(x) + (b << 23)); }

// data of the lane's owner slot j, in registers
template <class R>
struct JData {
    R ux, uy, uz, ia, fa, dfa, e0;
};

#ifndef F2_MINB_128
#define F2_MINB_128 20       // warps per SM asked of the 128-slot instantiation: 10 CTAs of 2 warps (96 registers, 21.7 KB each)
#endif
#ifndef F2_MINB1
#define F2_MINB1 20          // resident CTAs per SM asked of the one-warp-per-centre instantiation (metals: 5.2 vs 5.65 ms at 14)
#endif
template <class Spec, int WPC, int CAPA, bool TINY, class R>
__device__ __forceinline__ void force2_centre(const Force2Params& p, const int64_t i, unsigned char* smem_raw) {
    using R2 = typename Vec2<R>::type;
    constexpr int NT = WPC * 32;
    constexpr bool REGC = Spec::NACC <= 12;          // coefficients of the current group in registers
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    int tc = 0;
    for (int e = 1; e < p.n_elem; ++e)
        if (i >= p.cell_start[(size_t)e * p.ncell]) tc = e;
    if (p.variant[tc] != Spec::ID && !(Spec::FREE_ETA && p.variant[tc] == ANG_MULTI)) return;          // uniform per CTA
    const ElemProgram* __restrict__ prog = p.prog[tc];
    // free-eta kernels: one launch per pass (nnp_internal.h AngPass); the forces are additive over the passes
    const AngPass* __restrict__ ps = &prog->pass[Spec::FREE_ETA ? p.pass : 0];
    if (Spec::FREE_ETA && (p.pass >= prog->n_pass || ps->spec != Spec::ID)) return;
    const bool own_rc = Spec::FREE_ETA && ps->own_rc != 0;          // the pass's cutoff is shorter than the neighbour list's
    const bool widep = Spec::FREE_ETA && ps->wide != 0;             // wide angular functions: no r_jk term, every pair counts
    const int z0 = Spec::FREE_ETA ? ps->zeta0 : 1;                  // menu bits 0, 1, 2 stand for zeta = z0, 2 z0, 4 z0 ...
    const int zx = Spec::FREE_ETA ? ps->zeta_x : 16;                // ... and bit 4 for zeta = zx (16 z0: two more squarings)
    const bool zx_own = Spec::FREE_ETA && zx != 16 * z0;
    const double rc2p = Spec::FREE_ETA ? ps->rc2 : p.rc2, k2p = Spec::FREE_ETA ? ps->k2 : p.k2;
    const int32_t* __restrict__ n_ang = Spec::FREE_ETA ? ps->n_ang : prog->n_ang;
    const int neta = Spec::FREE_ETA ? ps->n_eta : Spec::NETA;
    const bool first_pass = !Spec::FREE_ETA || p.pass == 0;         // the radial forces
    const bool handover = !Spec::FREE_ETA || (prog->n_pass == 1 && !own_rc && !widep);   // masks from the SF kernel

    constexpr int capa = CAPA;
    const int npair = p.n_elem * (p.n_elem + 1) / 2;
    R2* p0 = reinterpret_cast<R2*>(smem_raw);               // (ux, uy)
    R2* p1 = p0 + capa;                                     // (uz, 1/a)
    R2* p2 = p1 + capa;                                     // (fc(a), fc'(a)/a)
    R2* acc0 = p2 + capa;                                   // WPC x (fxy[capa] R2, fz[capa] R, pad)
    SlotAcc2<R> acc;
    acc.fxy = acc0 + (size_t)wid * 2 * capa;
    acc.fz = reinterpret_cast<R*>(acc.fxy + capa);
    R* e0 = reinterpret_cast<R*>(acc0 + (size_t)WPC * 2 * capa);   // exp(-eta_0 a^2)
    R* rad = e0 + capa;                                       // radial scalar R
    GroupTab* tab = reinterpret_cast<GroupTab*>(reinterpret_cast<double*>(rad + capa + (capa & 1)));   // 8-byte aligned for R = float too
    R2* bt = reinterpret_cast<R2*>(tab + npair);              // [pair][bt2_stride] pairs of c_b = beta_b 2^(1-zeta_b)
    R* btc = reinterpret_cast<R*>(bt);                        // the same table, entry by entry
    int* wsum = reinterpret_cast<int*>(bt + npair * bt2_stride<Spec>());   // 16 ints of scratch
    double* brow = reinterpret_cast<double*>(wsum + 16);
    uint2* words = reinterpret_cast<uint2*>(brow + ((p.g_stride + 1) & ~1));   // (mask, descriptor)
    float4* f32 = reinterpret_cast<float4*>(acc0);            // alias: screening copy (dead before the accumulators are zeroed)
    uint16_t* C = reinterpret_cast<uint16_t*>(acc0 + capa);   // alias: prefix of the mask popcounts

    int seg[MAX_ELEM + 1];
    seg[0] = 0;
#pragma unroll
    for (int e = 0; e < MAX_ELEM; ++e) seg[e + 1] = seg[e] + p.nbr_cnt[(size_t)i * MAX_ELEM + e];
    const int ntot = seg[MAX_ELEM];
    if (ntot < p.nt_lo || ntot > p.nt_hi) return;   // uniform per CTA: another slot-capacity instantiation owns this centre

    for (int s = tid; s < p.g_stride; s += NT) brow[s] = p.dEdG[(size_t)i * p.g_stride + s];
    // The SF kernel has screened this centre already (Workspace::gmask): fetch its mask words now, so that
    // the global-memory latency hides behind the staging below (consumed after the group table exists).
#ifndef F2_NPRE
#define F2_NPRE 6
#endif
    constexpr int NPRE = F2_NPRE;                             // words per thread kept in registers
    const int64_t moff = p.word_off[i];
    const int nwg = (int)(p.word_off[i + 1] - moff);
    const bool have_masks = handover && moff + nwg <= p.gmask_cap;
    uint32_t pre[NPRE];
#pragma unroll
    for (int r = 0; r < NPRE; ++r) pre[r] = (have_masks && tid + r * NT < nwg) ? p.gmask[moff + tid + r * NT] : 0u;
    __syncthreads();

    // ---- stage the neighbourhood; radial part R = sum_r beta_r exp(-eta d^2) (fc'(a) - 2 eta d fc(a)) / a
    const double xi = p.sx[i], yi = p.sy[i], zi = p.sz[i];
    const int32_t* row = p.nbr + (size_t)i * p.stride;
    const double eta0 = prog->ang_eta[0];
    constexpr bool tiny = TINY;                      // exp(-eta_0 r^2) without range reduction (mathfn.cuh exp_tiny)
    if ((prog->tiny_exp != 0) != TINY) return;       // uniform per CTA: the other instantiation owns this element
    // radial forces: first pass only; with cutoff radii per symmetry function (ElemProgram::per_sf_rc) they are left to
    // the generic kernel's radial-only mode (k_force.cu) -- this kernel stages ONE fc per neighbour
    const bool radial_here = first_pass && prog->per_sf_rc == 0;
    for (int e = 0; e < p.n_elem; ++e) {
        const int nr = radial_here ? prog->n_rad[e] : 0, off = prog->rad_off[e];
        for (int m = seg[e] + tid; m < seg[e + 1]; m += NT) {
            const int j = row[m];
            const double dx = min_image_1d(xi, p.sx[j], p.box[0], p.half[0]);
            const double dy = min_image_1d(yi, p.sy[j], p.box[1], p.half[1]);
            const double dz = min_image_1d(zi, p.sz[j], p.box[2], p.half[2]);
            const double a2 = fma(dx, dx, fma(dy, dy, dz * dz));
            const double ia = rsqrt(a2);
            const double a = a2 * ia;
            const bool in = !own_rc || a2 < rc2p;               // beyond the pass's radius: fc = 0, and out of the screening
            double Ca = 0.0, Sa = 0.0;
            if (in) cos_sinc(a2 * k2p, Ca, Sa);
            const double fa = Ca * Ca;                          // fc(a)
            const double dfa_a = (-2.0 * k2p) * (Ca * Sa);      // fc'(a)/a
            p0[m] = mk2((R)dx, (R)dy);
            p1[m] = mk2((R)dz, (R)ia);
            p2[m] = mk2((R)fa, (R)dfa_a);
            e0[m] = (R)(Spec::FREE_ETA ? a2 : (tiny ? exp_tiny(-eta0 * a2) : exp_small(-eta0 * a2)));   // FREE_ETA: a^2 itself
            f32[m] = in ? make_float4((float)dx, (float)dy, (float)dz, 0.f) : make_float4(1e9f * (float)(m + 1), 0.f, 0.f, 0.f);
            double Rs = 0.0;
            for (int r = 0; r < nr; ++r) {
                const RadialSF f = prog->rad[off + r];
                const double d = a - f.rs;
                const double ex = exp_small(fmax(-f.eta * d * d, -700.0));
                Rs = fma(brow[f.g] * ex, fma(-2.0 * f.eta * d, fa * ia, dfa_a), Rs);
            }
            rad[m] = (R)Rs;
        }
    }
    // coefficient tables of all pair groups
    if (tid < 16) {
        for (int pr = 0; pr < npair; ++pr) {
#pragma unroll
            for (int e = 0; e < Spec::NETA; ++e) {
                if (Spec::mask(e) >> tid & 1u) {
                    const int g = Spec::FREE_ETA ? ps->g[pr][e][tid] : prog->ang_g[pr][e][tid];
                    const int zeta = (tid & 7) == Spec::MAXBIT ? zx : z0 << (tid & 7);
                    const double lam = tid < 8 ? 1.0 : -1.0;
                    const double bc = g >= 0 ? brow[g] * exp2((double)(1 - zeta)) : 0.0;
                    int a = 0;   // accumulator slot = set bits before (e, tid)
                    for (int ee = 0; ee < Spec::NETA; ++ee) {
                        const unsigned mk = Spec::mask(ee);
                        if (ee < e) a += __popc(mk);
                        else if (ee == e) a += __popc(mk & ((1u << tid) - 1u));
                    }
                    btc[pr * 2 * bt2_stride<Spec>() + a] = (R)bc;
                    (void)zeta; (void)lam;
                }
            }
        }
    }
    int NW = 0;
    const int ng = build_groups<true>(seg, p.n_elem, n_ang, tab, tid, NW);
    __syncthreads();

    // ---- screening -> masks; prefix; even split of the triplet stream over the NT threads ------------
    const float rc2f = widep ? 3.0e38f : (float)(rc2p * (1.0 + 1e-5));      // wide: no screening (a switched-off slot has fc = 0)
    if (have_masks) {
        // masks arrive in the SF kernel's group-major order; place them j-major and rebuild the descriptors
#pragma unroll
        for (int r = 0; r < NPRE; ++r) {
            const int y = tid + r * NT;
            if (y < NW) {
                int g, jl, w;
                decode_gmajor(tab, ng, y, g, jl, w);
                words[tab[g].woff + jl * tab[g].stride + w] = make_uint2(pre[r], word_desc(tab[g], jl, w));
            }
        }
        for (int y = tid + NPRE * NT; y < NW; y += NT) {
            int g, jl, w;
            decode_gmajor(tab, ng, y, g, jl, w);
            words[tab[g].woff + jl * tab[g].stride + w] = make_uint2(p.gmask[moff + y], word_desc(tab[g], jl, w));
        }
    } else {
        for (int g = 0; g < ng; ++g) screen_group(tab[g], f32, words, rc2f, tid, NT);
    }
    __syncthreads();
    const int T = mask_prefix(words, C, NW, tid, NT, wsum);
    __syncthreads();
    const int quota = (T + NT - 1) / NT;
    Walker wk;
    wk.words = words;
    wk.cnt = max(0, min(quota, T - tid * quota));
    wk.m = 1u; wk.d = 0u; wk.idx = 0;
    if (wk.cnt > 0) wk.seek(C, NW, tid * quota);
    __syncthreads();
    for (int m = tid; m < WPC * 2 * capa; m += NT) acc0[m] = mk2((R)0, (R)0);   // the aliases are dead
    __syncthreads();

    // ---- angular part: every lane walks its range of the stream ---------------------------------------
    R eta[Spec::NETA];
#pragma unroll
    for (int e = 0; e < Spec::NETA; ++e) eta[e] = (R)(Spec::FREE_ETA ? ps->eta[e] : prog->ang_eta[e]);
    const R eta0r = (R)eta0, k2r = (R)k2p, rc2r = (R)rc2p, m2k2 = (R)(-2.0 * k2p);
    JData<R> J;
    J.ux = J.uy = J.uz = (R)1; J.ia = (R)1; J.fa = (R)0; J.dfa = (R)0; J.e0 = (R)1;
    int jcur = -1, paircur = -1;
    R Aj = (R)0, Vx = (R)0, Vy = (R)0, Vz = (R)0;
    R cf[REGC ? Spec::NACC : 1];                      // c_b of the lane's current pair group
#pragma unroll
    for (int a = 0; a < (REGC ? Spec::NACC : 1); ++a) cf[a] = (R)0;
    uint32_t dcur = 0xffffffffu;
    for (int it = 0; it < quota; ++it) {
        const bool active = wk.cnt > 0;
        wk.advance();
        // New mask word: maybe a new owner slot (fold the j-side sums into the slot accumulator, load the
        // new j) and maybe a new pair group (reload the coefficients).  No conflict is possible inside the
        // loop: the stream is j-major, so the lanes that share a slot j are consecutive and only the last
        // of them leaves j before its range ends (the others flush after the loop).
        if (active && wk.d != dcur) {
            dcur = wk.d;
            const int jn = wk.j();
            if (jn != jcur) {
                if (jcur >= 0) {
                    R2 a = acc.fxy[jcur];
                    R b = acc.fz[jcur];
                    a.x += fma(-Aj, J.ux, Vx); a.y += fma(-Aj, J.uy, Vy); b += fma(-Aj, J.uz, Vz);
                    acc.fxy[jcur] = a;
                    acc.fz[jcur] = b;
                }
                jcur = jn;
                const R2 a0 = p0[jcur], a1 = p1[jcur], a2 = p2[jcur];
                J.ux = a0.x; J.uy = a0.y; J.uz = a1.x; J.ia = a1.y; J.fa = a2.x; J.dfa = a2.y; J.e0 = e0[jcur];
                Aj = (R)0; Vx = (R)0; Vy = (R)0; Vz = (R)0;
            }
            const int pr = p.n_elem <= 2 ? wk.pair2() : pair_of_slots(jn, wk.first_partner(), seg, p.n_elem);
            if (pr != paircur) {
                paircur = pr;
                if constexpr (REGC) {
                    const R2* src = reinterpret_cast<const R2*>(btc + pr * 2 * bt2_stride<Spec>());
#pragma unroll
                    for (int a = 0; a < Spec::NACC / 2; ++a) {
                        const R2 c = src[a];
                        cf[2 * a] = c.x; cf[2 * a + 1] = c.y;
                    }
                    if constexpr (Spec::NACC & 1) cf[Spec::NACC - 1] = btc[pr * 2 * bt2_stride<Spec>() + Spec::NACC - 1];
                }
            }
        }
        __syncwarp();
        // c_b of the lane's pair group: registers (REGC) or, for the large sets, 128-bit loads of c pairs per eta
        const R2* btg = bt + max(paircur, 0) * bt2_stride<Spec>();
        const int k = active ? wk.pop() : max(jcur, 0);
        const int rank = conflict_rank(k, active, lane);       // issued early: its latency hides behind the FP64 work
        const R2 k0 = p0[k], k1 = p1[k], k2v = p2[k];
        const R ek = e0[k];
        const R wx = k0.x - J.ux, wy = k0.y - J.uy, wz = k1.x - J.uz;
        const R c2 = fma(wx, wx, fma(wy, wy, wz * wz));
        R Cc, Sc;
        cos_sinc(c2 * k2r, Cc, Sc);
        R fcc = Cc * Cc;                               // fc(c)
        R dfc = m2k2 * (Cc * Sc);                      // fc'(c)/c
        if (widep) { fcc = (R)1; dfc = (R)0; }         // wide: no fc(c)
        if (!active || (!widep && !(c2 < rc2r))) { fcc = (R)0; dfc = (R)0; }   // cutoff (FP64: exact; the masks were screened in FP32)
        R Y[Spec::NETA];
        const R r2 = widep ? J.e0 + ek : (J.e0 + ek) + c2;       // FREE_ETA: a^2 + b^2 (+ c^2, narrow) -- the staged value is a^2
        if constexpr (!Spec::FREE_ETA) {
            // (exp_tiny5: degree 5, 1e-14 -- one DFMA per triplet less than the symmetry-function kernel's degree 6; 74.8 -> 73.9 ms)
            Y[0] = (J.e0 * ek) * (tiny ? exp_tiny5(-eta0r * c2) : exp_small(-eta0r * c2));
            if constexpr (Spec::NETA > 1) Y[1] = ipow<Spec::ratio(1)>(Y[Spec::rbase(1)]);
            if constexpr (Spec::NETA > 2) Y[2] = ipow<Spec::ratio(2)>(Y[Spec::rbase(2)]);
            if constexpr (Spec::NETA > 3) Y[3] = ipow<Spec::ratio(3)>(Y[Spec::rbase(3)]);
        }
        const R iab = J.ia * k1.y;
        const R cosv = fma(J.ux, k0.x, fma(J.uy, k0.y, J.uz * k1.x)) * iab;
        // pw[l][b] = (1 +- cos)^(2^b) ; pd[l][b] = (1 +- cos)^(2^b - 1)  (REGC: times zeta = 2^b)
        R pw[2][Spec::MAXBIT + 1], pd[2][Spec::MAXBIT + 1];
        pw[0][0] = (R)1 + cosv; pw[1][0] = (R)1 - cosv;
        pd[0][0] = (R)1; pd[1][0] = (R)1;
        const R base0 = pw[0][0], base1 = pw[1][0];
        if (Spec::FREE_ETA && z0 > 1) {                        // uniform per CTA: P = (1 +- cos)^z0, dP/d(1 +- cos) = z0 (1 +- cos)^(z0-1)
            const R q0 = powi_uniform(pw[0][0], z0 - 1), q1 = powi_uniform(pw[1][0], z0 - 1);
            pw[0][0] *= q0; pw[1][0] *= q1;
            pd[0][0] = (R)z0 * q0; pd[1][0] = (R)z0 * q1;
        }
#pragma unroll
        for (int b = 1; b <= Spec::MAXBIT; ++b) {
#pragma unroll
            for (int l = 0; l < 2; ++l) {
                pw[l][b] = pw[l][b - 1] * pw[l][b - 1];
                pd[l][b] = pd[l][b - 1] * pw[l][b - 1];
            }
        }
#pragma unroll
        for (int b = 1; b <= Spec::MAXBIT; ++b) {       // times zeta = 2^b: dP/dcos comes from the SAME coefficients
            pd[0][b] = scale2(pd[0][b], b);
            pd[1][b] = scale2(pd[1][b], b);
        }
        if (zx_own) {                                          // uniform per CTA: the top menu entry is an exponent of its own
            const R q0 = powi_uniform(base0, zx - 1), q1 = powi_uniform(base1, zx - 1);
            pw[0][Spec::MAXBIT] = base0 * q0; pw[1][Spec::MAXBIT] = base1 * q1;
            pd[0][Spec::MAXBIT] = (R)zx * q0; pd[1][Spec::MAXBIT] = (R)zx * q1;
        }
        R Z0 = (R)0, Z1 = (R)0, Z2 = (R)0;
#pragma unroll
        for (int e = 0; e < Spec::NETA; ++e) {
            if (Spec::FREE_ETA && e >= neta) break;            // uniform per CTA: eta slots the table does not use
            if constexpr (Spec::FREE_ETA) Y[e] = exp_small(-eta[e] * r2);
            R T0 = (R)0, T1 = (R)0;
            // the coefficients of eta_e sit at consecutive (even-aligned) accumulator indices
            constexpr int NE = 16;
            R ce[REGC ? 1 : NE];
            if constexpr (!REGC) {
                const int base = acc_index<Spec>(e, 0) & ~1;
#pragma unroll
                for (int q = 0; q < NE / 2; ++q) {
                    if (base + 2 * q < acc_index<Spec>(e + 1, 0)) {          // folds after unrolling: only this eta's pairs
                        const R2 v = btg[(base >> 1) + q];
                        ce[2 * q] = v.x; ce[2 * q + 1] = v.y;
                    } else { ce[2 * q] = (R)0; ce[2 * q + 1] = (R)0; }
                }
            }
#pragma unroll
            for (int b = 0; b <= Spec::MAXBIT; ++b) {
#pragma unroll
                for (int l = 0; l < 2; ++l)
                    if (Spec::mask(e) >> (8 * l + b) & 1u) {
                        R c;
                        if constexpr (REGC) c = cf[acc_index<Spec>(e, 8 * l + b)];
                        else c = ce[acc_index<Spec>(e, 8 * l + b) - (acc_index<Spec>(e, 0) & ~1)];
                        T0 = fma(c, pw[l][b], T0);
                        T1 = l == 0 ? fma(c, pd[l][b], T1) : fma(-c, pd[l][b], T1);
                    }
            }
            const R A = T0 * Y[e];
            Z0 += A;
            Z1 = fma(T1, Y[e], Z1);
            Z2 = fma(eta[e], A, Z2);
        }
        // slot scalars
        const R fab = J.fa * k2v.x;
        const R Cf = fab * fcc;
        const R t2 = (Cf + Cf) * Z2;
        const R f_w = widep ? (R)0 : fma(fab * dfc, Z0, -t2);      // wide: nothing depends on w
        const R q = Z1 * Cf;
        const R qc = q * cosv;
        const R f_uu = fma(-qc, J.ia * J.ia, fma((J.dfa * k2v.x) * fcc, Z0, -t2));
        const R f_vv = fma(-qc, k1.y * k1.y, fma((J.fa * k2v.y) * fcc, Z0, -t2));
        const R s1 = f_uu + f_w, s2 = f_vv + f_w, s3 = fma(-q, iab, f_w);
        Aj += s1;
        Vx = fma(s3, k0.x, Vx);
        Vy = fma(s3, k0.y, Vy);
        Vz = fma(s3, k1.x, Vz);
        // F_k = s3 u - s2 v
        slot_add(acc, k, active, rank, fma(s3, J.ux, -s2 * k0.x), fma(s3, J.uy, -s2 * k0.y), fma(s3, J.uz, -s2 * k1.x));
    }
    // the lanes whose ranges end inside the same slot j fold it in here, one after the other
    slot_add(acc, jcur, jcur >= 0, conflict_rank(jcur, jcur >= 0, lane), fma(-Aj, J.ux, Vx), fma(-Aj, J.uy, Vy),
             fma(-Aj, J.uz, Vz));
    __syncthreads();

    // ---- flush: F_slot - R u; one global FP64 RED per component; the centre gets minus the sum -------
    double fx = 0.0, fy = 0.0, fz = 0.0;
    for (int m = tid; m < ntot; m += NT) {
        const int j = row[m];
        const R2 u0 = p0[m];
        const R uz = p1[m].x;
        R2 fxy = acc0[m];
        R fzz = reinterpret_cast<const R*>(acc0 + capa)[m];
#pragma unroll
        for (int w = 1; w < WPC; ++w) {
            const R2 a = acc0[(size_t)w * 2 * capa + m];
            fxy.x += a.x; fxy.y += a.y;
            fzz += reinterpret_cast<const R*>(acc0 + (size_t)w * 2 * capa + capa)[m];
        }
        const double Rm = (double)rad[m];
        const double ax = fma(-Rm, (double)u0.x, (double)fxy.x), ay = fma(-Rm, (double)u0.y, (double)fxy.y),
                     az = fma(-Rm, (double)uz, (double)fzz);
        force_add(p, 3 * (size_t)j + 0, ax);
        force_add(p, 3 * (size_t)j + 1, ay);
        force_add(p, 3 * (size_t)j + 2, az);
        fx -= ax; fy -= ay; fz -= az;
    }
    fx = warp_sum(fx); fy = warp_sum(fy); fz = warp_sum(fz);
    if (lane == 0) {
        force_add(p, 3 * (size_t)i + 0, fx);
        force_add(p, 3 * (size_t)i + 1, fy);
        force_add(p, 3 * (size_t)i + 2, fz);
    }
}

#ifndef F2_MINB_F32
#define F2_MINB_F32 32       // warps per SM asked of the FP32 instantiations (mixed-precision mode)
#endif
template <class Spec, int WPC, int CAPA, class R>
__host__ __device__ constexpr int f2_min_blocks() {
    // 10 CTAs per SM only where the coefficients live in registers (NACC <= 12): the wide set at 96 registers
    // spilled into the loop (configs[4]: 10.38 vs 9.80 ms)
    return WPC == 1 ? F2_MINB1 : (sizeof(R) == 4 ? F2_MINB_F32 : (CAPA <= 128 && Spec::NACC <= 12 ? F2_MINB_128 : 14)) / WPC;
}

// one CTA per centre: blockIdx.x = sorted position of the centre
template <class Spec, int WPC, int CAPA, bool TINY, class R>
__global__ void __launch_bounds__(WPC * 32, f2_min_blocks<Spec, WPC, CAPA, R>()) k_force2(const __grid_constant__ Force2Params p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    force2_centre<Spec, WPC, CAPA, TINY, R>(p, (int64_t)blockIdx.x, smem_raw);
}

// the centres of a list (Workspace::big_list: those with more than 128 neighbours), a few CTAs walking it
template <class Spec, int WPC, int CAPA, bool TINY, class R>
__global__ void __launch_bounds__(WPC * 32, 14 / WPC) k_force2_list(const __grid_constant__ Force2Params p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n_list = *p.big_count;
    for (int q = blockIdx.x; q < n_list; q += gridDim.x) {
        force2_centre<Spec, WPC, CAPA, TINY, R>(p, (int64_t)p.big_list[q], smem_raw);
        __syncthreads();                             // the next centre reuses the shared memory
    }
}

#ifndef NNP_F2_WPC
#define NNP_F2_WPC 2
#endif
constexpr int F2_WPC = NNP_F2_WPC;

template <class Spec, int CAPA, bool TINY, class R, int WPC = F2_WPC>
static int launch_capa(Force2Params p, int nt_lo, int nt_hi, cudaStream_t st) {
    p.nt_lo = nt_lo; p.nt_hi = nt_hi;
    const size_t smem = force2_smem<Spec>(CAPA, p.g_stride, p.n_elem, WPC, sizeof(R));
    static unsigned long long configured = 0ull;      // per device (opt_in_smem)
    opt_in_smem(k_force2<Spec, WPC, CAPA, TINY, R>, &configured);
    k_force2<Spec, WPC, CAPA, TINY, R><<<(unsigned)p.n, WPC * 32, smem, st>>>(p);
    return 1;
}

template <class Spec, int CAPA, bool TINY, class R, int WPC = F2_WPC>
static int launch_capa_list(Force2Params p, int nt_lo, int nt_hi, cudaStream_t st) {
    p.nt_lo = nt_lo; p.nt_hi = nt_hi;
    const size_t smem = force2_smem<Spec>(CAPA, p.g_stride, p.n_elem, WPC, sizeof(R));
    static unsigned long long configured = 0ull;
    opt_in_smem(k_force2_list<Spec, WPC, CAPA, TINY, R>, &configured);
    const unsigned grid = (unsigned)(p.n < 148 * 8 ? p.n : 148 * 8);
    k_force2_list<Spec, WPC, CAPA, TINY, R><<<grid, WPC * 32, smem, st>>>(p);
    return 1;
}

// slot capacity = smallest instantiated CAPA that holds max_neighbors (nnp_set_max_neighbors: 32..255)
template <class Spec, bool TINY, class R = double>
static int launch_one2(const Force2Params& p, cudaStream_t st) {
    // small neighbourhoods (metals: ~20 neighbours, ~60 triplets per centre): 64 slots, ONE warp per centre (FP64 only)
    if (p.cap <= 64) return launch_capa<Spec, 64, TINY, double, 1>(p, 0, 64, st);
    // The 128-slot instantiation keeps 10 CTAs per SM resident (21.7 KB, 96 registers) against 8 of the 160-slot one
    // (27.5 KB, 119 registers): every centre with at most 128 neighbours runs on it (measured on configs[3]: 79.4 ->
    // 76.8 ms), the few others (water-like systems: 1 centre in ~10^4; listed by k_count_words) on a list-driven launch
    // of the bigger instantiation -- a second launch over all N centres costs 1.3 ms in CTAs that return at once.
    int launches = launch_capa<Spec, 128, TINY, R>(p, 0, 128, st);
    if (p.cap > 128) launches += p.cap <= 160 ? launch_capa_list<Spec, 160, TINY, R>(p, 129, 160, st)
                                              : launch_capa_list<Spec, 256, TINY, double>(p, 129, 255, st);
    return launches;
}

// launches the fast kernels for the specialised variants in use; the caller has zeroed f_sorted
int launch_force2(const Workspace& w, const Grid& g, int64_t n, int n_elem, const ElemProgram* const* d_prog,
                  const int* variant, const PassInfo& passes, double rc, int stride, int max_nbr, int g_stride, int precision,
                  cudaStream_t st) {
    if (n == 0) return 0;
    Force2Params p;
    p.n = n; p.n_elem = n_elem; p.ncell = g.ncell; p.stride = stride; p.cap = max_nbr; p.g_stride = g_stride; p.pass = 0;
    p.rc = rc; p.rc2 = rc * rc;
    p.k2 = (3.14159265358979323846 / (2.0 * rc)) * (3.14159265358979323846 / (2.0 * rc));
    for (int c = 0; c < 3; ++c) { p.box[c] = g.box[c]; p.half[c] = g.half[c]; }
    p.sx = w.sx; p.sy = w.sy; p.sz = w.sz;
    p.cell_start = w.cell_start; p.nbr = w.nbr; p.nbr_cnt = w.nbr_cnt; p.dEdG = w.dEdG; p.f_sorted = w.f_sorted;
    p.fixed = passes.fixed_forces; p.status = w.status; p.sticky = w.sticky;
    p.word_off = w.word_off; p.gmask = w.gmask; p.gmask_cap = w.gmask_cap;
    p.big_list = w.big_list; p.big_count = w.status + 2;
    bool use[ANG_NVARIANT][2] = {};                                       // [variant][tiny_exp]
    for (int e = 0; e < MAX_ELEM; ++e) {
        p.prog[e] = e < n_elem ? d_prog[e] : nullptr;
        p.variant[e] = e < n_elem ? (variant[e] & 255) : -1;                 // bit 8 of variant[] = tiny_exp of the element
        if (e < n_elem) use[variant[e] & 255][(variant[e] >> 8) & 1] = true;
    }
    int launches = 0;
    // precision 1 (nnp_set_precision: mixed): FP32 instantiations of BASELINE.json's two shapes, water-like exp range
    const bool f32 = precision == 1;
    if (max_nbr <= 32) {     // small neighbourhoods (metals): 8 lanes per centre (k_small.cu)
        if (use[ANG_BASE12][1]) launches += launch_force_small(w, g, n, n_elem, d_prog, variant, rc, stride, max_nbr, g_stride, true, passes.fixed_forces, st);
        if (use[ANG_BASE12][0]) launches += launch_force_small(w, g, n, n_elem, d_prog, variant, rc, stride, max_nbr, g_stride, false, passes.fixed_forces, st);
        use[ANG_BASE12][0] = use[ANG_BASE12][1] = false;
    }
    if (use[ANG_BASE12][1]) launches += f32 ? launch_one2<SpecBase12, true, float>(p, st) : launch_one2<SpecBase12, true>(p, st);
    if (use[ANG_BASE12][0]) launches += launch_one2<SpecBase12, false>(p, st);
    if (use[ANG_WIDE32][1]) launches += f32 ? launch_one2<SpecWide32, true, float>(p, st) : launch_one2<SpecWide32, true>(p, st);
    if (use[ANG_WIDE32][0]) launches += launch_one2<SpecWide32, false>(p, st);
    // free-eta tables: one launch per pass and kernel (the CTAs of elements without that pass return at once)
    for (int q = 0; q < MAX_PASS; ++q) {
        bool f32p = false, f16p = false;
        for (int e = 0; e < n_elem; ++e)
            if (q < passes.n_pass[e]) { f32p |= passes.spec[e][q] == ANG_FREE32; f16p |= passes.spec[e][q] == ANG_FREE16; }
        p.pass = q;
        if (f32p) launches += launch_one2<SpecFree32, false>(p, st);
        if (f16p) launches += launch_one2<SpecFree16, false>(p, st);
    }
    return launches;
}

}  // namespace nnp

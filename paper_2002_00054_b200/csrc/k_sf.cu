// k_sf.cu -- S2: atom-centred symmetry functions G_i (PAPER.md L40 step 1: radial descriptors,
// plus "a similar angular computation with one extra loop over neighbors of neighbors";
// formulas: include/nnp.h at nnp_sf, readings 2-4).
//
// GENERIC path: any symmetry-function table (walks the SF list per triplet).  Tables with the
// structure of a compile-time Spec (angular.cuh) run on the lane-owned fast path, k_sf2.cu.
// One warp per centre.  Radial and angular parts share the staged neighbourhood, so they are
// ONE kernel here (the paper splits them, L98, because its parallel_for has no shared staging).
#include "angular.cuh"
#include "geometry.cuh"

namespace nnp {

constexpr int SF_WARPS = 4;

struct SfParams {
    int64_t n;
    int n_elem, ncell, stride, cap, g_stride;
    int na_max;                          // largest angular pair group of the model (per-lane accumulators)
    double rc, rc2, inv_rc, k2;          // k2 = (pi / (2 rc))^2
    double box[3], half[3];
    const double *sx, *sy, *sz;
    const int32_t *cell_start, *nbr, *nbr_cnt;
    double* G;
    const ElemProgram* prog[MAX_ELEM];
    int variant[MAX_ELEM];
    int radial_only[MAX_ELEM];           // 1: run only the radial block for this element (per-SF radial radii of a lane-owned element)
};

template <class Spec>
__host__ __device__ constexpr size_t sf_warp_smem(int cap, int na_max) {
    // p0, p1, p2 (double2 each), a (double), FP32 screening copy (12 B) per slot; queue (64 x u32);
    // generic accumulators: one per (SF of the current pair group, lane)
    const size_t capa = (size_t)((cap + 3) & ~3);
    return capa * (48 + 8 + 12) + 256 + (Spec::ID == ANG_GENERIC ? (size_t)(na_max > 1 ? na_max : 1) * 32 * 8 : 0);
}

// ---- per-triplet work, generic group: walk the SF list, reduce each value over the batch -----
struct SfTripletGeneric {
    const Nbh& nb;
    const AngularSF* sf;
    int nsf;
    double k2, rc2;
    const double* ra; // [slot] distance a
    double* gacc;     // [nsf][32] per warp, shared memory: every lane sums its own triplets, reduced once per group
    int lane;
    bool own;         // the SFs carry their own cutoff radii (ElemProgram::per_sf_rc)

    __device__ __forceinline__ void operator()(int j, int k, int, bool active) {
        const double2 j0 = nb.p0[j], j1 = nb.p1[j], j2 = nb.p2[j];
        const double2 k0 = nb.p0[k], k1 = nb.p1[k], kq = nb.p2[k];
        const double wx = k0.x - j0.x, wy = k0.y - j0.y, wz = k1.x - j1.x;
        const double c2 = fma(wx, wx, fma(wy, wy, wz * wz));
        const double Cc = cos_only(c2 * k2);
        double Cw = j2.y * kq.y;                    // wide SFs (kind 9): fc(a) fc(b), no r_jk cutoff
        double C = Cw * (Cc * Cc);                  // narrow SFs: times fc(c), needs c < rc
        if (!active) Cw = 0.0;
        if (!active || !(c2 < rc2)) C = 0.0;
        const double cosv = (j0.x * k0.x + j0.y * k0.y + j1.x * k1.x) * (j1.y * k1.y);
        const double aj = ra[j], ak = ra[k];
        const double r2ab = aj * aj + ak * ak;
        const double r2sum = r2ab + c2;
        const double a2j = fma(j0.x, j0.x, fma(j0.y, j0.y, j1.x * j1.x)), a2k = fma(k0.x, k0.x, fma(k0.y, k0.y, k1.x * k1.x));
        // exp(-eta r^2) is shared by consecutive SFs of equal eta (the usual order of a table)
        double en = -1.0, ew = -1.0, Yn = 0.0, Yw = 0.0;
        for (int s = 0; s < nsf; ++s) {
            const AngularSF f = sf[s];
            if (own) {          // fc(.; rc_s) of this SF for a, b (and c)
                Cw = active ? fc_own(a2j, f.rc2, f.k2) * fc_own(a2k, f.rc2, f.k2) : 0.0;
                C = f.wide ? 0.0 : Cw * fc_own(c2, f.rc2, f.k2);
            }
            const double base = 1.0 + (double)f.lam * cosv;
            double pw = 1.0, bb = base;
            for (int z = f.izeta; z > 0; z >>= 1) {
                if (z & 1) pw *= bb;
                bb *= bb;
            }
            double v;
            if (f.wide) {
                if (f.eta != ew) { ew = f.eta; Yw = exp_small(fmax(-f.eta * r2ab, -700.0)); }
                v = f.coef * pw * Yw * Cw;
            } else {
                if (f.eta != en) { en = f.eta; Yn = exp_small(fmax(-f.eta * r2sum, -700.0)); }
                v = f.coef * pw * Yn * C;
            }
            gacc[s * 32 + lane] += v;
        }
        __syncwarp();
    }
};

template <class Spec>
__global__ void __launch_bounds__(SF_WARPS * 32) k_sf(const __grid_constant__ SfParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t i = (int64_t)blockIdx.x * SF_WARPS + wid;
    if (i >= p.n) return;
    int tc = 0;
    for (int e = 1; e < p.n_elem; ++e)
        if (i >= p.cell_start[(size_t)e * p.ncell]) tc = e;
    // radial_only: an element of the lane-owned kernels whose RADIAL functions carry their own cutoff radii -- those
    // kernels then leave the radial block to this one (they stage one fc per neighbour), the angular part stays theirs
    const bool radial_only = p.radial_only[tc] != 0;
    if (p.variant[tc] != Spec::ID && !radial_only) return;
    const ElemProgram* __restrict__ prog = p.prog[tc];

    const int capa = (p.cap + 3) & ~3;
    unsigned char* base = smem_raw + (size_t)wid * sf_warp_smem<Spec>(p.cap, p.na_max);
    Nbh nb;
    nb.p0 = reinterpret_cast<double2*>(base);
    nb.p1 = nb.p0 + capa;
    nb.p2 = nb.p1 + capa;
    nb.p3 = nullptr;
    double* ra = reinterpret_cast<double*>(nb.p2 + capa);
    nb.fxy = reinterpret_cast<float2*>(ra + capa);
    nb.fz = reinterpret_cast<float*>(nb.fxy + capa);
    PairQueue Q;
    Q.q = reinterpret_cast<uint32_t*>(nb.fz + capa);
    Q.head = 0;
    Q.n = 0;
    double* gacc = reinterpret_cast<double*>(Q.q + 64);

    // segment boundaries of the neighbour row (grouped by element)
    int seg[MAX_ELEM + 1];
    seg[0] = 0;
#pragma unroll
    for (int e = 0; e < MAX_ELEM; ++e) seg[e + 1] = seg[e] + p.nbr_cnt[(size_t)i * MAX_ELEM + e];
    const int ntot = seg[MAX_ELEM];

    // ---- stage the neighbourhood -------------------------------------------------------------
    const double xi = p.sx[i], yi = p.sy[i], zi = p.sz[i];
    const int32_t* row = p.nbr + (size_t)i * p.stride;
    double eta0 = 0.0;
    if constexpr (Spec::NETA > 0) eta0 = prog->ang_eta[0];
    for (int m = lane; m < ntot; m += 32) {
        const int j = row[m];
        const double dx = min_image_1d(xi, p.sx[j], p.box[0], p.half[0]);
        const double dy = min_image_1d(yi, p.sy[j], p.box[1], p.half[1]);
        const double dz = min_image_1d(zi, p.sz[j], p.box[2], p.half[2]);
        const double a2 = fma(dx, dx, fma(dy, dy, dz * dz));
        const double ia = rsqrt(a2);
        const double Ca = cos_only(a2 * p.k2);
        double E0 = 0.0;
        if constexpr (Spec::NETA > 0) E0 = exp_small(-eta0 * a2);
        nb.p0[m] = make_double2(dx, dy);
        nb.p1[m] = make_double2(dz, ia);
        nb.p2[m] = make_double2(E0, Ca * Ca);       // (exp(-eta_0 a^2), fc(a))
        ra[m] = a2 * ia;
        nb.fxy[m] = make_float2((float)dx, (float)dy);
        nb.fz[m] = (float)dz;
    }
    __syncwarp();

    double* Grow = p.G + (size_t)i * p.g_stride;
    if (!radial_only)
        for (int s = prog->n_sf + lane; s < p.g_stride; s += 32) Grow[s] = 0.0;

    // ---- radial: G = sum_j exp(-eta (a - rs)^2) fc(a) over the neighbours of element e ----------
    for (int e = 0; e < p.n_elem; ++e) {
        const int nr = prog->n_rad[e], off = prog->rad_off[e];
        for (int r = 0; r < nr; ++r) {
            const RadialSF f = prog->rad[off + r];
            double acc = 0.0;
            for (int m = seg[e] + lane; m < seg[e + 1]; m += 32) {
                const double d = ra[m] - f.rs;
                double fcv = nb.p2[m].y;
                if (prog->per_sf_rc) {
                    const double2 u0 = nb.p0[m];
                    const double uz = nb.p1[m].x;
                    fcv = fc_own(fma(u0.x, u0.x, fma(u0.y, u0.y, uz * uz)), f.rc2, f.k2);
                }
                acc = fma(exp_small(fmax(-f.eta * d * d, -700.0)), fcv, acc);
            }
            acc = warp_sum(acc);
            if (lane == 0) Grow[f.g] = acc;
        }
    }

    if (radial_only) return;                          // warp-uniform
    // ---- angular groups -----------------------------------------------------------------------
    const float rc2f = screen_rc2(p.rc2);
    for (int e1 = 0; e1 < p.n_elem; ++e1)
        for (int e2 = e1; e2 < p.n_elem; ++e2) {
            const int pr = pair_index(e1, e2, p.n_elem);
            const int na = prog->n_ang[pr];
            if (na == 0) continue;
            {
                for (int s = 0; s < na; ++s) gacc[s * 32 + lane] = 0.0;
                __syncwarp();
                SfTripletGeneric f{nb, prog->ang + prog->ang_off[pr], na, p.k2, p.rc2, ra, gacc, lane, prog->per_sf_rc != 0};
                const float rs = group_has_wide(prog->ang + prog->ang_off[pr], na) ? 3.0e38f : rc2f;   // wide SFs: no r_jk screen
                if (e1 == e2) pairs_within(nb, seg[e1], seg[e1 + 1] - seg[e1], rs, Q, lane, f);
                else pairs_between(nb, seg[e1], seg[e1 + 1] - seg[e1], seg[e2], seg[e2 + 1] - seg[e2], rs, Q, lane, f);
                __syncwarp();
                for (int s = 0; s < na; ++s) {
                    const double v = warp_sum(gacc[s * 32 + lane]);
                    if (lane == 0) Grow[prog->ang[prog->ang_off[pr] + s].g] = v;
                }
                __syncwarp();
            }
        }
}

template <class Spec>
static int launch_one(const SfParams& p, cudaStream_t st) {
    const size_t smem = SF_WARPS * sf_warp_smem<Spec>(p.cap, p.na_max);
    static unsigned long long configured = 0ull;      // per device (opt_in_smem)
    opt_in_smem(k_sf<Spec>, &configured);
    const unsigned nb = (unsigned)((p.n + SF_WARPS - 1) / SF_WARPS);
    k_sf<Spec><<<nb, SF_WARPS * 32, smem, st>>>(p);
    return 1;
}

int launch_sf(const Workspace& w, const Grid& g, int64_t n, int n_elem, const ElemProgram* const* d_prog,
              const int* variant, const PassInfo& passes, double rc, int stride, int max_nbr, int g_stride, int na_max,
              int precision, cudaStream_t st) {
    if (n == 0) return 0;
    SfParams p;
    p.na_max = na_max;
    p.n = n; p.n_elem = n_elem; p.ncell = g.ncell; p.stride = stride; p.cap = max_nbr; p.g_stride = g_stride;
    p.rc = rc; p.rc2 = rc * rc; p.inv_rc = 1.0 / rc;
    p.k2 = (3.14159265358979323846 / (2.0 * rc)) * (3.14159265358979323846 / (2.0 * rc));
    for (int c = 0; c < 3; ++c) { p.box[c] = g.box[c]; p.half[c] = g.half[c]; }
    p.sx = w.sx; p.sy = w.sy; p.sz = w.sz;
    p.cell_start = w.cell_start; p.nbr = w.nbr; p.nbr_cnt = w.nbr_cnt; p.G = w.G;
    bool use[ANG_NVARIANT] = {};
    for (int e = 0; e < MAX_ELEM; ++e) {
        p.prog[e] = e < n_elem ? d_prog[e] : nullptr;
        p.variant[e] = e < n_elem ? (variant[e] & 255) : -1;      // bit 8 = tiny_exp flag (fast launchers)
        p.radial_only[e] = (e < n_elem && (variant[e] & 255) != ANG_GENERIC && passes.radial_own[e]) ? 1 : 0;
        if (e < n_elem) use[variant[e] & 255] = true;
        if (p.radial_only[e]) use[ANG_GENERIC] = true;
    }
    int launches = 0;
    if (use[ANG_BASE12] || use[ANG_WIDE32] || use[ANG_FREE32] || use[ANG_FREE16] || use[ANG_MULTI])     // specialised tables: lane-owned design (k_sf2.cu)
        launches += launch_sf2(w, g, n, n_elem, d_prog, variant, passes, rc, stride, max_nbr, g_stride, precision, st);
    if (use[ANG_GENERIC]) launches += launch_one<SpecGeneric>(p, st);
    return launches;
}

}  // namespace nnp

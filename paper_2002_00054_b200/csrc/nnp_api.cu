// nnp_api.cu -- the C ABI of libnnp_b200 (include/nnp.h): model construction, workspace layout,
// the nnp_compute pipeline S0..S5, the host-buffer entry point and the debug exports.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "angular.cuh"
#include "nnp_internal.h"

using namespace nnp;

struct nnp_model {
    int n_elem = 0;
    std::vector<std::string> names;
    double rc = 0.0;
    int device = 0;
    int max_nbr = 160;
    int precision = 0;              // NNP_PRECISION_F64 / NNP_PRECISION_MIXED (nnp_set_precision)
    int g_stride = 0;
    int na_max = 0;                 // largest angular pair group (SF count) of any element
    int n_sf_elem[MAX_ELEM] = {0, 0, 0, 0};
    ElemProgram* d_prog[MAX_ELEM] = {nullptr, nullptr, nullptr, nullptr};
    std::vector<ElemProgram> h_prog;             // host copies as built by nnp_create (global rc, specialised variants)
    std::vector<std::pair<int, int>> sf_loc;     // per SF of the nnp_create table: (central element, position in its G)
    int variant[MAX_ELEM] = {0, 0, 0, 0};
    PassInfo passes = {};            // free-eta passes per element, force-accumulation mode (launchers)
    NetDesc nets[MAX_ELEM];
    double* d_weights[MAX_ELEM] = {nullptr, nullptr, nullptr, nullptr};
    double* d_scaling[MAX_ELEM] = {nullptr, nullptr, nullptr, nullptr};
    MlpRegWeights* reg_w[MAX_ELEM] = {nullptr, nullptr, nullptr, nullptr};   // host, see NetDesc::reg
    cudaGraphExec_t md_exec = nullptr;     // graph of one MD step of the last nnp_md_run (kept until the next run)
    cudaStream_t md_exec_stream = nullptr;   // [2][n_sf]: shift, scale (or null)
    // last nnp_compute (for the exports)
    Workspace ws;
    bool have_ws = false;
    int64_t last_n = 0;
    cudaStream_t last_stream = nullptr;
    int last_launches = 0;
    int32_t* h_status = nullptr;   // pinned
    int32_t* d_sticky = nullptr;   // device word: OR of the status flags of every call since the last nnp_sync_status
    // neighbour-skin mode (nnp_set_neighbor_skin): what the candidate list in the caller's workspace was built for
    double skin = 0.0;
    int32_t* d_skin_stats = nullptr;   // [2]: calls, rebuilds
    bool skin_valid = false;
    void* skin_ws = nullptr;
    int64_t skin_n = 0;
    double skin_box[3] = {0.0, 0.0, 0.0};
    // timing
    bool timing = false;
    bool timing_valid = false;
    cudaEvent_t ev[NNP_N_STAGES + 1];
    bool ev_created = false;
    // host-buffer path
    cudaStream_t hstream = nullptr;
    void* h_ws = nullptr;
    size_t h_ws_bytes = 0;
    int64_t h_cap = 0;
    double *hd_pos = nullptr, *hd_e = nullptr, *hd_f = nullptr, *hd_etot = nullptr;
    int32_t* hd_type = nullptr;
    std::string err;
};

static thread_local std::string g_create_err = "";   // nnp_last_error(NULL): per host thread

// (pi / (2 rc))^2, the argument scale of the cutoff polynomials (same arithmetic as the kernel launchers)
static double k2_of(double rc) {
    const double t = 3.14159265358979323846 / (2.0 * rc);
    return t * t;
}

static void set_pass_info(nnp_model* m, const std::vector<ElemProgram>& progs) {
    const int fixed = m->passes.fixed_forces;
    std::memset(&m->passes, 0, sizeof(m->passes));
    m->passes.fixed_forces = fixed;
    for (int c = 0; c < m->n_elem; ++c) {
        m->passes.n_pass[c] = progs[c].n_pass;
        m->passes.radial_own[c] = progs[c].per_sf_rc;
        for (int q = 0; q < progs[c].n_pass; ++q) m->passes.spec[c][q] = progs[c].pass[q].spec;
    }
}

static nnp_status fail(nnp_model* m, nnp_status s, const std::string& msg) {
    if (m) m->err = msg;
    else g_create_err = msg;
    return s;
}

#define NNP_CUDA(m, expr)                                                                       \
    do {                                                                                        \
        cudaError_t e__ = (expr);                                                               \
        if (e__ != cudaSuccess)                                                                 \
            return fail(m, NNP_ERR_CUDA, std::string(#expr) + ": " + cudaGetErrorString(e__)); \
    } while (0)

struct DeviceGuard {
    int prev = -1;
    bool ok;
    explicit DeviceGuard(int dev) {
        ok = cudaGetDevice(&prev) == cudaSuccess && cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard() {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

// ---------------------------------------------------------------- workspace layout

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

static size_t ws_layout(Workspace* w, void* base, int64_t n, int n_elem, int stride, int g_stride, int sstride) {
    size_t off = 0;
    auto take = [&](size_t bytes) -> void* {
        void* p = base ? (void*)((char*)base + off) : nullptr;
        off = align_up(off + bytes, 256);
        return p;
    };
    const size_t N = (size_t)(n > 0 ? n : 1);
    w->sx = (double*)take(N * 8); w->sy = (double*)take(N * 8); w->sz = (double*)take(N * 8);
    w->tx = (double*)take(N * 8); w->ty = (double*)take(N * 8); w->tz = (double*)take(N * 8);
    w->perm = (int32_t*)take(N * 4); w->tperm = (int32_t*)take(N * 4);
    w->key = (int32_t*)take(N * 4); w->rank = (int32_t*)take(N * 4); w->tkey = (int32_t*)take(N * 4);
    w->n_keys_cap = (int64_t)n_elem * (2 * (int64_t)N + 64) + 1;
    w->cell_start = (int32_t*)take((size_t)w->n_keys_cap * 4);
    w->scan_tmp_len = w->n_keys_cap / 2048 + 16384;
    w->scan_tmp = (int32_t*)take((size_t)w->scan_tmp_len * 4);
    w->nbr = (int32_t*)take(N * (size_t)stride * 4);
    w->nbr_cnt = (int32_t*)take(N * MAX_ELEM * 4);
    w->snbr = nullptr; w->snbr_cnt = nullptr; w->bx = w->by = w->bz = nullptr; w->skin_flag = nullptr; w->skin_stats = nullptr;
    if (sstride > 0) {
        w->snbr = (int32_t*)take(N * (size_t)sstride * 4);
        w->snbr_cnt = (int32_t*)take(N * MAX_ELEM * 4);
        w->bx = (double*)take(N * 8); w->by = (double*)take(N * 8); w->bz = (double*)take(N * 8);
        w->skin_flag = (int32_t*)take(64);
    }
    w->slist = stride <= 32 ? (uint16_t*)take(N * (size_t)SMALL_LIST_U16 * 2) : nullptr;
    w->G = (double*)take(N * (size_t)g_stride * 8);
    w->dEdG = (double*)take(N * (size_t)g_stride * 8);
    w->e_sorted = (double*)take(N * 8);
    w->f_sorted = (double*)take(N * 3 * 8);
    w->big_list = (int32_t*)take(N * 4);
    w->nw = (int32_t*)take(N * 4);
    w->word_off = (int64_t*)take((N + 1) * 8);
    w->word_tmp = (int64_t*)take(((N + 1) / 4096 + 2 * 4096 + 16) * 8);
    w->gmask_cap = (int64_t)N * WORD_BUDGET;
    w->gmask = (uint32_t*)take((size_t)w->gmask_cap * 4);
    w->n_partial = (int64_t)(N + 255) / 256 + 1;
    w->partial = (double*)take((size_t)w->n_partial * 8);
    w->status = (int32_t*)take(64);
    w->bytes = off;
    return off;
}

static bool make_grid(Grid* g, const double box[3], double rc, int64_t n) {
    const int64_t limit = 2 * (n > 0 ? n : 1) + 64;
    for (int hw = 2; hw >= 1; --hw) {
        const double cs_min = rc * (1.0 + 1e-9) / hw;   // margin: a cell index rounded the wrong way must not hide a neighbour
        double nc[3];
        for (int c = 0; c < 3; ++c) {
            nc[c] = std::floor(box[c] / cs_min);
            if (nc[c] < 1.0) nc[c] = 1.0;
        }
        // cells of rc/2 pay when they hold a few atoms each (one warp per cell, nnp_internal.h Grid)
        if (hw == 2 && (double)n < 1.5 * nc[0] * nc[1] * nc[2]) continue;
        while (nc[0] * nc[1] * nc[2] > (double)limit) {
            const double s = std::cbrt((double)limit / (nc[0] * nc[1] * nc[2])) * 0.999;
            for (int c = 0; c < 3; ++c) nc[c] = std::fmax(1.0, std::floor(nc[c] * s));
        }
        g->hw = hw;
        for (int c = 0; c < 3; ++c) {
            g->box[c] = box[c];
            g->half[c] = 0.5 * box[c];
            g->nc[c] = (int)nc[c];
            g->inv_cs[c] = nc[c] / box[c];
            g->span[c] = g->nc[c] >= 2 * hw + 1 ? hw : 0;
        }
        g->ncell = g->nc[0] * g->nc[1] * g->nc[2];
        return true;
    }
    return false;
}

// ---------------------------------------------------------------- create / destroy

// try to express the angular groups of one element on a specialised variant
template <class Spec>
static bool match_spec(const std::vector<std::vector<AngularSF>>& groups, ElemProgram* P) {
    std::vector<double> etas;
    for (const auto& grp : groups)
        for (const auto& f : grp) {
            bool seen = false;
            for (double e : etas) seen |= (e == f.eta);
            if (!seen) etas.push_back(f.eta);
        }
    if ((int)etas.size() != Spec::NETA) return false;
    for (size_t a = 0; a < etas.size(); ++a)
        for (size_t b = a + 1; b < etas.size(); ++b)
            if (etas[b] < etas[a]) std::swap(etas[a], etas[b]);
    if (!(etas[0] > 0.0)) return false;
    for (int e = 1; e < Spec::NETA; ++e) {
        const double want = etas[Spec::rbase(e)] * Spec::ratio(e);
        if (std::fabs(etas[e] - want) > 1e-12 * want) return false;
    }
    for (int e = 0; e < MAX_ETA; ++e) P->ang_eta[e] = e < Spec::NETA ? etas[e] : 0.0;
    for (size_t p = 0; p < groups.size(); ++p) {
        for (int e = 0; e < MAX_ETA; ++e)
            for (int b = 0; b < 16; ++b) P->ang_g[p][e][b] = -1;
        if (groups[p].empty()) continue;
        unsigned seen[MAX_ETA] = {0, 0, 0, 0};
        for (const auto& f : groups[p]) {
            int e = -1;
            for (int q = 0; q < Spec::NETA; ++q)
                if (etas[q] == f.eta) e = q;
            int bit = -1;
            for (int b = 0; b < 7; ++b)
                if (f.izeta == (1 << b)) bit = b;
            if (e < 0 || bit < 0) return false;
            if (f.lam < 0) bit += 8;
            if (!(Spec::mask(e) >> bit & 1u) || (seen[e] >> bit & 1u)) return false;
            seen[e] |= 1u << bit;
            P->ang_g[p][e][bit] = (int16_t)f.g;
        }
        for (int e = 0; e < Spec::NETA; ++e)
            if (seen[e] != Spec::mask(e)) return false;
    }
    return true;
}

// Free-eta passes (nnp_internal.h AngPass): any table of angular symmetry functions (narrow, kind 3, and wide, kind 9)
// with lambda = +-1, integer zeta and no (kind, rc, eta, lambda, zeta) twice in a pair group.  The symmetry functions
// are split by kind, cutoff radius and EXPONENT MENU (zeta0, zeta_x): the kernels' menu of a pass holds the exponents
// {zeta0, 2 zeta0, 4 zeta0, zeta_x}.  Inside one (kind, radius) the smallest zeta not yet covered becomes the next zeta0;
// its zeta_x is 16 zeta0 if the table has it (the kernels then square on), else the smallest zeta still uncovered (raised
// by square-and-multiply).  {1, 2, 4, 16}, {1, 4} and {1, 2, 3, 4} are one menu each.  Inside one such class the eta values
// go in chunks of at most four of about equal size; one pass per chunk, narrow first, radius descending.  Returns false if
// the table does not fit (more than MAX_PASS passes, an exponent beyond exp_small's range).
static bool build_passes(const std::vector<std::vector<AngularSF>>& groups, double rc, ElemProgram* P) {
    struct Key { double rc2, eta, k2; int wide, z0, zx; };
    static_assert((SpecFree32::mask(0) & 0xffu) == 0x17u && (SpecFree16::mask(0) & 0xffu) == 0x17u, "menu bits 0, 1, 2, 4");
    auto menu_bit = [](int zeta, int z0, int zx) {                  // menu bit of zeta in the menu (z0, zx), else -1
        for (int b = 0; b < 3; ++b)
            if (zeta == (z0 << b)) return b;
        return zeta == zx ? 4 : -1;
    };
    // menus per (kind, radius): the zeta values of the class in ascending order, see above
    struct Cls { double rc2; int wide; std::vector<int> zetas, z0, zx; };
    std::vector<Cls> classes;
    for (const auto& grp : groups)
        for (const auto& f : grp) {
            if (f.eta * 3.0 * f.rc2 > 700.0) return false;
            Cls* c = nullptr;
            for (auto& q : classes)
                if (q.rc2 == f.rc2 && q.wide == f.wide) c = &q;
            if (!c) { classes.push_back(Cls{f.rc2, f.wide, {}, {}, {}}); c = &classes.back(); }
            bool have = false;
            for (int z : c->zetas) have |= z == f.izeta;
            if (!have) c->zetas.push_back(f.izeta);
        }
    if (classes.empty()) return false;
    for (auto& c : classes) {
        std::sort(c.zetas.begin(), c.zetas.end());
        std::vector<int> open = c.zetas;                            // not yet on a menu, ascending
        auto take = [&](int z) {
            for (size_t q = 0; q < open.size(); ++q)
                if (open[q] == z) { open.erase(open.begin() + q); return true; }
            return false;
        };
        // No menu entry, used or not, may overflow: (1 +- cos) <= 2 and the kernels compute EVERY entry of a menu (an unused one
        // has coefficient 0, and 0 * inf is NaN), in FP32 in the mixed-precision mode.  So zeta0 <= 16 (4 zeta0 <= 64), the
        // squaring to 16 zeta0 only for zeta0 <= 4, and a larger exponent goes to the zeta_x entry of a menu with zeta0 = 1.
        while (!open.empty()) {
            int z0 = open.front(), zx;
            if (z0 > 16) {
                zx = z0; z0 = 1;
                take(zx);
            } else {
                take(z0); take(2 * z0); take(4 * z0);
                zx = 16 * z0;
                if (!(z0 <= 4 && take(zx))) {
                    if (!open.empty()) { zx = open.front(); take(zx); }
                    else if (z0 > 4) zx = z0;                       // unused: a harmless repeat of zeta0
                }
            }
            c.z0.push_back(z0);
            c.zx.push_back(zx);
        }
    }
    // the menu (index into its class) that holds a symmetry function
    auto menu_of = [&](const AngularSF& f, int& z0, int& zx) {
        for (const auto& c : classes)
            if (c.rc2 == f.rc2 && c.wide == f.wide)
                for (size_t q = 0; q < c.z0.size(); ++q)
                    if (menu_bit(f.izeta, c.z0[q], c.zx[q]) >= 0) { z0 = c.z0[q]; zx = c.zx[q]; return; }
        z0 = zx = 0;
    };
    std::vector<Key> keys;
    for (const auto& grp : groups)
        for (const auto& f : grp) {
            int z0, zx;
            menu_of(f, z0, zx);
            bool seen = false;
            for (const Key& k : keys) seen |= (k.rc2 == f.rc2 && k.eta == f.eta && k.wide == f.wide && k.z0 == z0 && k.zx == zx);
            if (!seen) keys.push_back(Key{f.rc2, f.eta, f.k2, f.wide, z0, zx});
        }
    auto before = [](const Key& a, const Key& b) {              // sort: narrow first, rc descending, zeta0 and eta ascending
        if (a.wide != b.wide) return a.wide < b.wide;
        if (a.rc2 != b.rc2) return a.rc2 > b.rc2;
        if (a.z0 != b.z0) return a.z0 < b.z0;
        if (a.zx != b.zx) return a.zx < b.zx;
        return a.eta < b.eta;
    };
    for (size_t x = 0; x < keys.size(); ++x)
        for (size_t y = x + 1; y < keys.size(); ++y)
            if (before(keys[y], keys[x])) std::swap(keys[x], keys[y]);
    int np = 0;
    size_t x = 0;
    while (x < keys.size()) {
        size_t y = x;
        while (y < keys.size() && keys[y].rc2 == keys[x].rc2 && keys[y].wide == keys[x].wide && keys[y].z0 == keys[x].z0 &&
               keys[y].zx == keys[x].zx) ++y;
        const int n = (int)(y - x), chunks = (n + MAX_ETA - 1) / MAX_ETA;
        for (int c = 0; c < chunks; ++c) {
            if (np >= MAX_PASS) return false;
            const int lo = (int)x + (n * c) / chunks, hi = (int)x + (n * (c + 1)) / chunks;
            AngPass& ps = P->pass[np++];
            std::memset(&ps, 0, sizeof(ps));
            ps.n_eta = hi - lo;
            for (int e = 0; e < MAX_ETA; ++e) ps.eta[e] = keys[lo + (e < ps.n_eta ? e : ps.n_eta - 1)].eta;
            ps.rc2 = keys[lo].rc2;
            ps.k2 = keys[lo].k2;                            // k2_of(rc_p), as stored with the symmetry function
            ps.own_rc = ps.rc2 != rc * rc ? 1 : 0;
            ps.wide = keys[lo].wide;
            ps.zeta0 = keys[lo].z0;
            ps.zeta_x = keys[lo].zx;
            ps.spec = ps.n_eta <= SpecFree16::NETA ? ANG_FREE16 : ANG_FREE32;
            for (size_t pr = 0; pr < groups.size(); ++pr) {
                for (int e = 0; e < MAX_ETA; ++e)
                    for (int b = 0; b < 16; ++b) ps.g[pr][e][b] = -1;
                for (const auto& f : groups[pr]) {
                    int fz0, fzx;
                    menu_of(f, fz0, fzx);
                    if (f.rc2 != ps.rc2 || f.wide != ps.wide || fz0 != ps.zeta0 || fzx != ps.zeta_x) continue;
                    int e = -1;
                    for (int q = ps.n_eta - 1; q >= 0; --q)
                        if (ps.eta[q] == f.eta) e = q;
                    if (e < 0) continue;
                    int bit = menu_bit(f.izeta, ps.zeta0, ps.zeta_x);
                    if (f.lam < 0) bit += 8;
                    if (ps.g[pr][e][bit] >= 0) return false;    // the same (rc, eta, lambda, zeta) twice in a pair group
                    ps.g[pr][e][bit] = (int16_t)f.g;
                    ps.n_ang[pr] += 1;
                }
            }
        }
        // (an in-kernel loop over the passes of one radius was measured: +7 % on single-pass tables for the loop structure,
        //  -3 % on a three-pass table -- the triplet loops dominate, not the staging)
        x = y;
    }
    P->n_pass = np;
    return true;
}

// Choice of kernels for one element from its complete program (lists, per-SF radii); nnp_create and
// nnp_set_sf_cutoffs both end here.  Sets variant, tiny_exp, per_sf_rc and the pass tables.
static nnp_status select_variant(ElemProgram& P, int n_elem, double rc, std::string& err) {
    const int npair = n_elem * (n_elem + 1) / 2;
    std::vector<std::vector<AngularSF>> groups(npair);
    bool own_ang = false, own_rad = false, any_ang = false;
    int nr = 0;
    for (int e = 0; e < n_elem; ++e) nr += P.n_rad[e];
    for (int r = 0; r < nr; ++r) own_rad |= P.rad[r].rc2 != rc * rc;
    for (int p = 0; p < npair; ++p)
        for (int a = 0; a < P.n_ang[p]; ++a) {
            groups[p].push_back(P.ang[P.ang_off[p] + a]);
            own_ang |= groups[p].back().rc2 != rc * rc;
            any_ang = true;
        }
    P.per_sf_rc = (own_ang || own_rad) ? 1 : 0;
    P.variant = ANG_GENERIC;
    P.n_pass = 0;
    P.tiny_exp = 0;
    if (!any_ang) return NNP_OK;
    // the specialised kernels use exp_small() unclamped: its argument -eta (a^2+b^2+c^2) must stay > -700
    double eta_max = 0.0;
    bool any_wide = false;           // wide angular SFs run on the generic kernels only
    for (int p = 0; p < npair; ++p)
        for (const auto& f : groups[p]) { eta_max = std::fmax(eta_max, f.eta); any_wide |= f.wide != 0; }
    const bool in_range = !any_wide && eta_max * 3.0 * rc * rc <= 700.0;
    if (in_range && !own_ang && match_spec<SpecBase12>(groups, &P)) P.variant = ANG_BASE12;
    else if (in_range && !own_ang && match_spec<SpecWide32>(groups, &P)) P.variant = ANG_WIDE32;
    else if (build_passes(groups, rc, &P))
        P.variant = (P.n_pass == 1 && !P.pass[0].own_rc && !P.pass[0].wide) ? P.pass[0].spec : ANG_MULTI;
    else {
        P.n_pass = 0;
        for (int p = 0; p < npair; ++p)
            if (P.n_ang[p] > 64) {
                err = "generic angular path supports <= 64 SFs per pair group";
                return NNP_ERR_LIMIT;
            }
    }
    P.tiny_exp = ((P.variant == ANG_BASE12 || P.variant == ANG_WIDE32) && P.ang_eta[0] * rc * rc * (1.0 + 1e-5) <= 0.05) ? 1 : 0;
    return NNP_OK;
}

// Host side of nnp_create: validate the SF table and build every element's program, including the choice of
// kernels (ElemProgram::variant).  No CUDA call in here -- nnp_table_kernels exposes the choice to CPU-only tests.
static nnp_status build_tables(int n_elem, double rc, int n_sf, const nnp_sf* sf, std::vector<ElemProgram>& progs,
                               int count[MAX_ELEM], int& na_max, std::string& err) {
    auto tfail = [&](const char* msg) {
        err = msg;
        return NNP_ERR_INVALID_ARG;
    };
    auto lfail = [&](const char* msg) {
        err = msg;
        return NNP_ERR_LIMIT;
    };
    na_max = 0;
    progs.assign(n_elem, ElemProgram());
    std::vector<std::vector<std::vector<AngularSF>>> ang(n_elem);   // [central][pair] -> list
    std::vector<std::vector<std::vector<RadialSF>>> rad(n_elem);    // [central][nbr element] -> list
    int npair = n_elem * (n_elem + 1) / 2;
    for (int c = 0; c < MAX_ELEM; ++c) count[c] = 0;
    for (int c = 0; c < n_elem; ++c) { ang[c].resize(npair); rad[c].resize(n_elem); }
    for (int q = 0; q < n_sf; ++q) {
        const nnp_sf& f = sf[q];
        if (f.central < 0 || f.central >= n_elem) return tfail("sf.central out of range");
        if (!(f.eta >= 0.0) || !std::isfinite(f.eta)) return tfail("sf.eta must be >= 0");
        const int g = count[f.central]++;
        if (f.kind == 2) {
            if (f.e1 < 0 || f.e1 >= n_elem) return tfail("sf.e1 out of range");
            if (!std::isfinite(f.rs)) return tfail("sf.rs not finite");
            rad[f.central][f.e1].push_back(RadialSF{f.eta, f.rs, g, 0, rc * rc, k2_of(rc)});
        } else if (f.kind == 3 || f.kind == 9) {
            if (f.e1 < 0 || f.e1 >= n_elem || f.e2 < 0 || f.e2 >= n_elem)
                return tfail("sf.e1/e2 out of range");
            if (!(f.lambda == 1.0 || f.lambda == -1.0))
                return tfail("angular lambda must be +1 or -1");
            const int iz = (int)f.zeta;
            if ((double)iz != f.zeta || iz < 1 || iz > 64)
                return tfail("angular zeta must be an integer in [1, 64]");
            const int a = f.e1 < f.e2 ? f.e1 : f.e2, b = f.e1 < f.e2 ? f.e2 : f.e1;
            ang[f.central][pair_index(a, b, n_elem)].push_back(
                AngularSF{f.eta, std::exp2(1.0 - f.zeta), g, iz, f.lambda > 0 ? 1 : -1, f.kind == 9 ? 1 : 0, rc * rc,
                          k2_of(rc)});
        } else {
            return tfail("sf.kind must be 2 (radial), 3 (angular narrow) or 9 (angular wide)");
        }
    }

    for (int c = 0; c < n_elem; ++c) {
        ElemProgram& P = progs[c];
        std::memset(&P, 0, sizeof(P));
        P.n_sf = count[c];
        P.n_elem = n_elem;
        if (count[c] < 1) return tfail("an element has no symmetry functions");
        int ro = 0;
        for (int e = 0; e < n_elem; ++e) {
            P.n_rad[e] = (int)rad[c][e].size();
            P.rad_off[e] = ro;
            if (ro + P.n_rad[e] > MAX_RAD_TOTAL) return lfail("more than 128 radial SFs for one element");
            for (const auto& f : rad[c][e]) P.rad[ro++] = f;
        }
        int ao = 0;
        for (int p = 0; p < npair; ++p) {
            P.n_ang[p] = (int)ang[c][p].size();
            if (P.n_ang[p] > na_max) na_max = P.n_ang[p];
            P.ang_off[p] = ao;
            if (ao + P.n_ang[p] > MAX_ANG_TOTAL) return lfail("more than 512 angular SFs for one element");
            for (const auto& f : ang[c][p]) P.ang[ao++] = f;
        }
        const nnp_status vs = select_variant(P, n_elem, rc, err);
        if (vs != NNP_OK) return vs;
    }
    return NNP_OK;
}

extern "C" nnp_status nnp_create(nnp_model** out, int32_t n_elem, const char* const* elem_names, double rc,
                                 int32_t n_sf, const nnp_sf* sf, const int32_t* n_layers,
                                 const int32_t* const* layer_sizes, const double* const* weights,
                                 int32_t cuda_device) {
    if (!out) return fail(nullptr, NNP_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (n_elem < 1) return fail(nullptr, NNP_ERR_INVALID_ARG, "n_elem must be >= 1");
    if (n_elem > MAX_ELEM) return fail(nullptr, NNP_ERR_LIMIT, "n_elem > NNP_MAX_ELEMENTS (4): this build keeps 4 element segments per neighbour row");
    if (!(rc > 0.0) || !std::isfinite(rc)) return fail(nullptr, NNP_ERR_INVALID_ARG, "rc must be > 0");
    if (n_sf < 1 || !sf || !n_layers || !layer_sizes || !weights)
        return fail(nullptr, NNP_ERR_INVALID_ARG, "null table");

    std::vector<ElemProgram> progs;
    int count[MAX_ELEM];
    int na_max_tab = 0;
    {
        std::string terr;
        const nnp_status ts = build_tables(n_elem, rc, n_sf, sf, progs, count, na_max_tab, terr);
        if (ts != NNP_OK) return fail(nullptr, ts, terr);
    }
    const int npair = n_elem * (n_elem + 1) / 2;
    (void)npair;

    nnp_model* m = new nnp_model();
    m->n_elem = n_elem;
    m->rc = rc;
    m->device = cuda_device;
    for (int c = 0; c < n_elem; ++c) m->names.push_back(elem_names && elem_names[c] ? elem_names[c] : "?");
    auto bail = [&](nnp_status s, const std::string& msg) {
        g_create_err = msg;
        nnp_destroy(m);
        return s;
    };

    m->na_max = na_max_tab;
    for (int c = 0; c < n_elem; ++c) {
        m->n_sf_elem[c] = count[c];
        if (count[c] > m->g_stride) m->g_stride = count[c];
        m->variant[c] = progs[c].variant | (progs[c].tiny_exp << 8);      // bit 8: host-side copy of tiny_exp for the launchers
    }

    // networks: validate and pack everything on the host first, upload afterwards
    std::vector<std::vector<double>> packed_all(n_elem);
    for (int c = 0; c < n_elem; ++c) {
        const int L = n_layers[c];
        if (L < 1) return bail(NNP_ERR_INVALID_ARG, "n_layers must be >= 1");
        if (L > MAX_LAYERS) return bail(NNP_ERR_LIMIT, "more than 8 weight layers");
        const int32_t* sz = layer_sizes[c];
        if (!sz || !weights[c]) return bail(NNP_ERR_INVALID_ARG, "null layer_sizes/weights");
        if (sz[0] != count[c]) return bail(NNP_ERR_INVALID_ARG, "first layer size must equal the element's SF count");
        if (sz[L] != 1) return bail(NNP_ERR_INVALID_ARG, "last layer size must be 1");
        NetDesc& nd = m->nets[c];
        std::memset(&nd, 0, sizeof(nd));
        nd.n_layers = L;
        for (int l = 0; l <= L; ++l) {
            if (sz[l] < 1) return bail(NNP_ERR_INVALID_ARG, "layer width < 1");
            if (l > 0 && l < L && sz[l] > MAX_WIDTH) return bail(NNP_ERR_LIMIT, "hidden layer wider than NNP_MAX_HIDDEN_WIDTH (256)");
            nd.sizes[l] = sz[l];
        }
        auto r4 = [](int x) { return (x + 3) & ~3; };
        size_t tot = 0;
        for (int l = 0; l < L; ++l) {
            nd.wt_off[l] = (int)tot; tot += (size_t)sz[l] * r4(sz[l + 1]);
            nd.w_off[l] = (int)tot; tot += (size_t)sz[l + 1] * r4(sz[l]);
            nd.b_off[l] = (int)tot; tot += (size_t)r4(sz[l + 1]);
        }
        std::vector<double> packed(tot, 0.0);
        const double* src = weights[c];
        for (int l = 0; l < L; ++l) {
            const int nin = sz[l], nout = sz[l + 1];
            const double* W = src;
            const double* B = src + (size_t)nin * nout;
            src = B + nout;
            for (int o = 0; o < nout; ++o)
                for (int i = 0; i < nin; ++i) {
                    const double v = W[(size_t)o * nin + i];
                    if (!std::isfinite(v)) return bail(NNP_ERR_INVALID_ARG, "non-finite weight");
                    packed[nd.wt_off[l] + (size_t)i * r4(nout) + o] = v;
                    packed[nd.w_off[l] + (size_t)o * r4(nin) + i] = v;
                }
            for (int o = 0; o < nout; ++o) packed[nd.b_off[l] + o] = B[o];
        }
        if (mlp_smem_bytes(nd, 8) > 200 * 1024) return bail(NNP_ERR_LIMIT, "network too large for the shared-memory tile");
        // parameter-block copy for the register kernel: n_in -> n1 -> n2 -> 1 with n1, n2 <= 32
        if (L == 3 && sz[1] <= MLP_REG_H && sz[2] <= MLP_REG_H &&
            (size_t)sz[0] * MLP_REG_H + 2 * MLP_REG_H + MLP_REG_H * MLP_REG_H + MLP_REG_H + 1 <= (size_t)MLP_REG_MAXW) {
            MlpRegWeights* R = new MlpRegWeights();
            std::memset(R, 0, sizeof(*R));
            R->n_in = sz[0]; R->n1 = sz[1]; R->n2 = sz[2];
            const int H = MLP_REG_H;
            const double* W1 = weights[c];
            const double* B1 = W1 + (size_t)sz[1] * sz[0];
            const double* W2 = B1 + sz[1];
            const double* B2 = W2 + (size_t)sz[2] * sz[1];
            const double* W3 = B2 + sz[2];
            const double* B3 = W3 + sz[2];
            double* q = R->w;
            for (int o = 0; o < sz[1]; ++o)
                for (int i = 0; i < sz[0]; ++i) q[(size_t)i * H + o] = W1[(size_t)o * sz[0] + i];
            q += (size_t)sz[0] * H;
            for (int o = 0; o < sz[1]; ++o) q[o] = B1[o];
            q += H;
            for (int o = 0; o < sz[2]; ++o)
                for (int i = 0; i < sz[1]; ++i) q[(size_t)i * H + o] = W2[(size_t)o * sz[1] + i];
            q += (size_t)H * H;
            for (int o = 0; o < sz[2]; ++o) q[o] = B2[o];
            q += H;
            for (int o = 0; o < sz[2]; ++o) q[o] = W3[o];
            q += H;
            q[0] = B3[0];
            m->reg_w[c] = R;
            nd.reg = R;
        }
        packed_all[c].swap(packed);
    }
    for (int c = 0; c < n_elem; ++c) {
        NetDesc& nd = m->nets[c];
        const std::vector<double>& packed = packed_all[c];
        const size_t tot = packed.size();
        DeviceGuard dg(cuda_device);
        if (!dg.ok) return bail(NNP_ERR_CUDA, "cudaSetDevice failed (no CUDA device?)");
        cudaError_t e = cudaMalloc(&m->d_weights[c], tot * sizeof(double));
        if (e == cudaSuccess) e = cudaMemcpy(m->d_weights[c], packed.data(), tot * sizeof(double), cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMalloc(&m->d_prog[c], sizeof(ElemProgram));
        if (e == cudaSuccess) e = cudaMemcpy(m->d_prog[c], &progs[c], sizeof(ElemProgram), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) return bail(NNP_ERR_CUDA, std::string("model upload: ") + cudaGetErrorString(e));
        nd.weights = m->d_weights[c];
    }
    {
        DeviceGuard dg(cuda_device);
        if (cudaMallocHost(&m->h_status, 64) != cudaSuccess) return bail(NNP_ERR_CUDA, "cudaMallocHost failed");
        std::memset(m->h_status, 0, 64);
        if (cudaMalloc(&m->d_sticky, 64) != cudaSuccess || cudaMemset(m->d_sticky, 0, 64) != cudaSuccess)
            return bail(NNP_ERR_CUDA, "cudaMalloc failed");
        m->d_skin_stats = m->d_sticky + 4;       // words 4, 5 of the same allocation
    }
    m->h_prog = progs;
    set_pass_info(m, progs);
    {
        int cnt[MAX_ELEM] = {0, 0, 0, 0};
        for (int s = 0; s < n_sf; ++s) m->sf_loc.push_back({sf[s].central, cnt[sf[s].central]++});
    }
    *out = m;
    return NNP_OK;
}

extern "C" void nnp_destroy(nnp_model* m) {
    if (!m) return;
    DeviceGuard dg(m->device);
    for (int c = 0; c < MAX_ELEM; ++c) {
        if (m->d_prog[c]) cudaFree(m->d_prog[c]);
        if (m->d_weights[c]) cudaFree(m->d_weights[c]);
        if (m->d_scaling[c]) cudaFree(m->d_scaling[c]);
        delete m->reg_w[c];
    }
    if (m->h_status) cudaFreeHost(m->h_status);
    if (m->d_sticky) cudaFree(m->d_sticky);
    if (m->ev_created)
        for (int k = 0; k <= NNP_N_STAGES; ++k) cudaEventDestroy(m->ev[k]);
    if (m->h_ws) cudaFree(m->h_ws);
    if (m->hd_pos) cudaFree(m->hd_pos);
    if (m->hd_type) cudaFree(m->hd_type);
    if (m->hd_e) cudaFree(m->hd_e);
    if (m->hd_f) cudaFree(m->hd_f);
    if (m->hd_etot) cudaFree(m->hd_etot);
    if (m->md_exec) { cudaStreamSynchronize(m->md_exec_stream); cudaGraphExecDestroy(m->md_exec); }
    if (m->hstream) cudaStreamDestroy(m->hstream);
    delete m;
}

extern "C" nnp_status nnp_table_kernels(int32_t n_elem, double rc, int32_t n_sf, const nnp_sf* sf, int32_t* kernels_out) {
    if (n_elem > MAX_ELEM) return fail(nullptr, NNP_ERR_LIMIT, "n_elem > NNP_MAX_ELEMENTS (4)");
    if (n_elem < 1 || !(rc > 0.0) || !std::isfinite(rc) || n_sf < 1 || !sf || !kernels_out)
        return fail(nullptr, NNP_ERR_INVALID_ARG, "bad table arguments");
    std::vector<ElemProgram> progs;
    int count[MAX_ELEM], na_max = 0;
    std::string terr;
    const nnp_status ts = build_tables(n_elem, rc, n_sf, sf, progs, count, na_max, terr);
    if (ts != NNP_OK) return fail(nullptr, ts, terr);
    for (int c = 0; c < n_elem; ++c) kernels_out[c] = progs[c].variant;
    return NNP_OK;
}

extern "C" nnp_status nnp_set_sf_cutoffs(nnp_model* m, int32_t n_sf, const double* h_rc) {
    if (!m) return NNP_ERR_INVALID_ARG;
    if (h_rc && n_sf != (int32_t)m->sf_loc.size()) return fail(m, NNP_ERR_INVALID_ARG, "n_sf differs from the table of nnp_create");
    std::vector<std::vector<double>> rcg(m->n_elem);
    for (int c = 0; c < m->n_elem; ++c) rcg[c].assign(m->n_sf_elem[c], m->rc);
    if (h_rc)
        for (size_t s = 0; s < m->sf_loc.size(); ++s) {
            if (!(h_rc[s] > 0.0) || !(h_rc[s] <= m->rc)) return fail(m, NNP_ERR_INVALID_ARG, "SF cutoff must be in (0, rc]");
            rcg[m->sf_loc[s].first][m->sf_loc[s].second] = h_rc[s];
        }
    const int npair = m->n_elem * (m->n_elem + 1) / 2;
    std::vector<ElemProgram> progs = m->h_prog;
    for (int c = 0; c < m->n_elem; ++c) {
        ElemProgram& P = progs[c];
        bool own = false;
        int nr = 0, na = 0;
        for (int e = 0; e < m->n_elem; ++e) nr += P.n_rad[e];
        for (int p = 0; p < npair; ++p) na += P.n_ang[p];
        for (int r = 0; r < nr; ++r) {
            const double x = rcg[c][P.rad[r].g];
            P.rad[r].rc2 = x * x;
            P.rad[r].k2 = k2_of(x);
            own |= x != m->rc;
        }
        for (int a = 0; a < na; ++a) {
            const double x = rcg[c][P.ang[a].g];
            P.ang[a].rc2 = x * x;
            P.ang[a].k2 = k2_of(x);
            own |= x != m->rc;
        }
        (void)own;
        // radii on angular symmetry functions: free-eta passes, one cutoff radius per pass, if the table fits them,
        // else the generic kernels; radii on radial functions only: the element keeps its kernels (their radial block
        // evaluates fc per symmetry function)
        std::string verr;
        const nnp_status vs = select_variant(P, m->n_elem, m->rc, verr);
        if (vs != NNP_OK) return fail(m, vs, verr);
    }
    DeviceGuard dg(m->device);
    if (!dg.ok) return fail(m, NNP_ERR_CUDA, "cudaSetDevice failed");
    NNP_CUDA(m, cudaDeviceSynchronize());          // the old tables may still be in use
    for (int c = 0; c < m->n_elem; ++c) {
        NNP_CUDA(m, cudaMemcpy(m->d_prog[c], &progs[c], sizeof(ElemProgram), cudaMemcpyHostToDevice));
        m->variant[c] = progs[c].variant | (progs[c].tiny_exp << 8);
    }
    set_pass_info(m, progs);
    return NNP_OK;
}

extern "C" nnp_status nnp_set_sf_scaling(nnp_model* m, int32_t elem, const double* h_shift, const double* h_scale) {
    if (!m) return NNP_ERR_INVALID_ARG;
    if (elem < 0 || elem >= m->n_elem) return fail(m, NNP_ERR_INVALID_ARG, "element index out of range");
    if ((h_shift == nullptr) != (h_scale == nullptr)) return fail(m, NNP_ERR_INVALID_ARG, "shift and scale go together");
    DeviceGuard dg(m->device);
    if (!dg.ok) return fail(m, NNP_ERR_CUDA, "cudaSetDevice failed");
    NNP_CUDA(m, cudaDeviceSynchronize());          // the old arrays may still be in use
    NetDesc& nd = m->nets[elem];
    if (m->d_scaling[elem]) { cudaFree(m->d_scaling[elem]); m->d_scaling[elem] = nullptr; }
    nd.sf_shift = nd.sf_scale = nullptr;
    if (!h_shift) return NNP_OK;
    const int n = m->n_sf_elem[elem];
    for (int s = 0; s < n; ++s)
        if (!std::isfinite(h_shift[s]) || !std::isfinite(h_scale[s])) return fail(m, NNP_ERR_INVALID_ARG, "non-finite scaling");
    NNP_CUDA(m, cudaMalloc(&m->d_scaling[elem], 2 * (size_t)n * sizeof(double)));
    NNP_CUDA(m, cudaMemcpy(m->d_scaling[elem], h_shift, n * sizeof(double), cudaMemcpyHostToDevice));
    NNP_CUDA(m, cudaMemcpy(m->d_scaling[elem] + n, h_scale, n * sizeof(double), cudaMemcpyHostToDevice));
    nd.sf_shift = m->d_scaling[elem];
    nd.sf_scale = m->d_scaling[elem] + n;
    return NNP_OK;
}

extern "C" nnp_status nnp_set_activation(nnp_model* m, int32_t kind) {
    if (!m) return NNP_ERR_INVALID_ARG;
    if (kind != NNP_ACT_SOFTPLUS && kind != NNP_ACT_TANH) return fail(m, NNP_ERR_INVALID_ARG, "unknown activation");
    for (int c = 0; c < m->n_elem; ++c) m->nets[c].activation = kind;
    return NNP_OK;
}

extern "C" nnp_status nnp_set_precision(nnp_model* m, int32_t mode) {
    if (!m) return NNP_ERR_INVALID_ARG;
    if (mode != NNP_PRECISION_F64 && mode != NNP_PRECISION_MIXED) return fail(m, NNP_ERR_INVALID_ARG, "unknown precision mode");
    m->precision = mode;
    return NNP_OK;
}

extern "C" nnp_status nnp_set_deterministic_forces(nnp_model* m, int32_t enabled) {
    if (!m) return NNP_ERR_INVALID_ARG;
    m->passes.fixed_forces = enabled != 0 ? 1 : 0;
    return NNP_OK;
}

extern "C" nnp_status nnp_set_max_neighbors(nnp_model* m, int32_t max_neighbors) {
    if (!m) return NNP_ERR_INVALID_ARG;
    if (max_neighbors < 16) return fail(m, NNP_ERR_INVALID_ARG, "max_neighbors must be >= 16");
    if (max_neighbors > NNP_MAX_NEIGHBORS)
        return fail(m, NNP_ERR_LIMIT, "max_neighbors > NNP_MAX_NEIGHBORS (255): the kernels address neighbour slots with 8 bits");
    m->max_nbr = max_neighbors;
    m->have_ws = false;
    m->skin_valid = false;
    return NNP_OK;
}

extern "C" nnp_status nnp_set_neighbor_skin(nnp_model* m, double skin) {
    if (!m) return NNP_ERR_INVALID_ARG;
    if (!(skin >= 0.0) || !std::isfinite(skin)) return fail(m, NNP_ERR_INVALID_ARG, "skin must be finite and >= 0");
    if (skin > m->rc) return fail(m, NNP_ERR_INVALID_ARG, "skin > rc");
    DeviceGuard dg(m->device);
    if (!dg.ok) return fail(m, NNP_ERR_CUDA, "cudaSetDevice failed");
    if (m->have_ws) NNP_CUDA(m, cudaStreamSynchronize(m->last_stream));
    NNP_CUDA(m, cudaMemset(m->d_skin_stats, 0, 2 * sizeof(int32_t)));
    m->skin = skin;
    m->skin_valid = false;
    m->have_ws = false;              // the workspace layout changes
    return NNP_OK;
}

extern "C" nnp_status nnp_invalidate_neighbors(nnp_model* m) {
    if (!m) return NNP_ERR_INVALID_ARG;
    m->skin_valid = false;
    return NNP_OK;
}

extern "C" nnp_status nnp_get_neighbor_rebuilds(nnp_model* m, int64_t* n_calls, int64_t* n_rebuilds) {
    if (!m || !n_calls || !n_rebuilds) return NNP_ERR_INVALID_ARG;
    DeviceGuard dg(m->device);
    if (!dg.ok) return fail(m, NNP_ERR_CUDA, "cudaSetDevice failed");
    if (m->have_ws) NNP_CUDA(m, cudaStreamSynchronize(m->last_stream));
    int32_t h[2] = {0, 0};
    NNP_CUDA(m, cudaMemcpy(h, m->d_skin_stats, sizeof(h), cudaMemcpyDeviceToHost));
    *n_calls = h[0];
    *n_rebuilds = h[1];
    return NNP_OK;
}

static int row_stride(const nnp_model* m) { return (m->max_nbr + 7) & ~7; }
// neighbour-skin mode: capacity of a candidate row = max_neighbors scaled by the volume ratio of the two spheres, plus slack
static int skin_max(const nnp_model* m) {
    if (!(m->skin > 0.0)) return 0;
    const double r = (m->rc + m->skin) / m->rc;
    return (int)std::ceil(m->max_nbr * r * r * r) + 16;
}
static int skin_stride(const nnp_model* m) { return (skin_max(m) + 7) & ~7; }

extern "C" size_t nnp_workspace_bytes(const nnp_model* m, int64_t n_atoms) {
    if (!m || n_atoms < 0) return 0;
    Workspace w;
    return ws_layout(&w, nullptr, n_atoms, m->n_elem, row_stride(m), m->g_stride, skin_stride(m));
}

extern "C" int32_t nnp_g_stride(const nnp_model* m) { return m ? m->g_stride : 0; }
extern "C" int32_t nnp_last_launch_count(const nnp_model* m) { return m ? m->last_launches : 0; }
extern "C" int32_t nnp_uses_fast_path(const nnp_model* m) {
    if (!m) return 0;
    for (int c = 0; c < m->n_elem; ++c)
        if ((m->variant[c] & 255) == ANG_GENERIC) return 0;
    return 1;
}
extern "C" const char* nnp_last_error(const nnp_model* m) { return m ? m->err.c_str() : g_create_err.c_str(); }
extern "C" const char* nnp_version(void) { return "0.1"; }

// ---------------------------------------------------------------- compute

extern "C" nnp_status nnp_compute(nnp_model* m, int64_t n_atoms, const double* d_pos, const int32_t* d_type,
                                  const double box[3], double* d_e_atom, double* d_e_total, double* d_force,
                                  void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
    if (!m) return NNP_ERR_INVALID_ARG;
    if (n_atoms < 0 || n_atoms > 0x7fffffffLL / 4) return fail(m, NNP_ERR_INVALID_ARG, "n_atoms out of range");
    if (!box || !d_e_total) return fail(m, NNP_ERR_INVALID_ARG, "box / d_e_total is NULL");
    if (n_atoms > 0 && (!d_pos || !d_type || !d_e_atom || !d_force)) return fail(m, NNP_ERR_INVALID_ARG, "null array");
    for (int c = 0; c < 3; ++c) {
        if (!std::isfinite(box[c]) || !(box[c] > 0.0)) return fail(m, NNP_ERR_INVALID_ARG, "box length must be finite and > 0");
        if (box[c] < 2.0 * (m->rc + m->skin)) return fail(m, NNP_ERR_BOX_TOO_SMALL, "box length < 2*(rc + skin)");
    }
    const int stride = row_stride(m);
    Workspace w;
    const size_t need = ws_layout(&w, d_workspace, n_atoms, m->n_elem, stride, m->g_stride, skin_stride(m));
    if (!d_workspace || ((uintptr_t)d_workspace & 255u) || workspace_bytes < need)
        return fail(m, NNP_ERR_WORKSPACE, "workspace null, misaligned or too small");
    w.sticky = m->d_sticky;
    w.skin_stats = m->d_skin_stats;
    DeviceGuard dg(m->device);
    if (!dg.ok) return fail(m, NNP_ERR_CUDA, "cudaSetDevice failed");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    Grid g;
    make_grid(&g, box, m->rc + m->skin, n_atoms);
    // neighbour-skin mode: 1 = this call must rebuild (nothing valid in this workspace for this n and box), 2 = the device decides
    int skin_mode = 0;
    if (m->skin > 0.0)
        skin_mode = (m->skin_valid && m->skin_ws == d_workspace && m->skin_n == n_atoms && m->skin_box[0] == box[0] &&
                     m->skin_box[1] == box[1] && m->skin_box[2] == box[2]) ? 2 : 1;
    if (m->timing && !m->ev_created) {
        for (int k = 0; k <= NNP_N_STAGES; ++k) NNP_CUDA(m, cudaEventCreate(&m->ev[k]));
        m->ev_created = true;
    }
    auto mark = [&](int k) {
        if (m->timing) cudaEventRecord(m->ev[k], st);
    };
    int launches = 0;
    if (n_atoms == 0) {   // nothing to launch: E = 0
        NNP_CUDA(m, cudaMemsetAsync(d_e_total, 0, sizeof(double), st));
        NNP_CUDA(m, cudaMemsetAsync(w.status, 0, sizeof(int32_t) * 4, st));
        m->timing_valid = false;
        m->ws = w; m->have_ws = true; m->last_n = 0; m->last_stream = st; m->last_launches = 0;
        m->skin_valid = false;
        return NNP_OK;
    }
    mark(0);
    launches += launch_sort(w, g, n_atoms, m->n_elem, d_pos, d_type, skin_mode, m->skin, st);
    mark(1);
    launches += launch_neighbors(w, g, n_atoms, m->n_elem, m->rc * m->rc, stride, m->max_nbr, skin_mode,
                                 (m->rc + m->skin) * (m->rc + m->skin), skin_stride(m), skin_max(m), st);
    if (skin_mode) {
        m->skin_valid = true; m->skin_ws = d_workspace; m->skin_n = n_atoms;
        for (int c = 0; c < 3; ++c) m->skin_box[c] = box[c];
    }
    mark(2);
    launches += launch_word_offsets(w, g, n_atoms, m->n_elem, m->d_prog, st);
    launches += launch_sf(w, g, n_atoms, m->n_elem, m->d_prog, m->variant, m->passes, m->rc, stride, m->max_nbr, m->g_stride, m->na_max, m->precision, st);
    mark(3);
    launches += launch_mlp(w, n_atoms, m->n_elem, g.ncell, m->nets, m->g_stride, st);
    mark(4);
    launches += launch_force(w, g, n_atoms, m->n_elem, m->d_prog, m->variant, m->passes, m->rc, stride, m->max_nbr, m->g_stride, m->precision, st);
    mark(5);
    launches += launch_finalize(w, n_atoms, d_e_atom, d_e_total, d_force, m->passes.fixed_forces, st);
    mark(6);
    m->timing_valid = m->timing;
    m->ws = w;
    m->have_ws = true;
    m->last_n = n_atoms;
    m->last_stream = st;
    m->last_launches = launches;
    NNP_CUDA(m, cudaGetLastError());
    return NNP_OK;
}

extern "C" nnp_status nnp_md_run(nnp_model* m, int32_t n_steps, double dt_fs, const double* h_mass, int64_t n_atoms,
                                 double* d_pos, double* d_vel, const int32_t* d_type, const double box[3],
                                 double* d_e_atom, double* d_e_total, double* d_force, void* d_workspace,
                                 size_t workspace_bytes, void* cuda_stream) {
    if (!m) return NNP_ERR_INVALID_ARG;
    if (n_steps < 0 || !h_mass || !(dt_fs > 0.0) || !std::isfinite(dt_fs)) return fail(m, NNP_ERR_INVALID_ARG, "n_steps / dt / masses");
    for (int e = 0; e < m->n_elem; ++e)
        if (!(h_mass[e] > 0.0) || !std::isfinite(h_mass[e])) return fail(m, NNP_ERR_INVALID_ARG, "mass must be finite and > 0");
    if (n_atoms > 0 && (!d_pos || !d_vel || !d_type || !d_force)) return fail(m, NNP_ERR_INVALID_ARG, "null array");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int launches = 0;
    auto one_step = [&]() -> nnp_status {
        {
            DeviceGuard dg(m->device);
            if (!dg.ok) return fail(m, NNP_ERR_CUDA, "cudaSetDevice failed");
            launches += launch_vv(n_atoms, m->n_elem, h_mass, d_type, d_force, d_vel, d_pos, dt_fs, true, st);
        }
        const nnp_status rc = nnp_compute(m, n_atoms, d_pos, d_type, box, d_e_atom, d_e_total, d_force, d_workspace,
                                          workspace_bytes, cuda_stream);
        if (rc != NNP_OK) return rc;
        launches += m->last_launches;
        DeviceGuard dg(m->device);
        launches += launch_vv(n_atoms, m->n_elem, h_mass, d_type, d_force, d_vel, d_pos, dt_fs, false, st);
        return NNP_OK;
    };
    if (m->md_exec) {       // the graph of the previous run may still be executing
        DeviceGuard dg(m->device);
        cudaStreamSynchronize(m->md_exec_stream);
        cudaGraphExecDestroy(m->md_exec);
        m->md_exec = nullptr;
    }
    int done = 0;
    // A step is 16 launches with fixed arguments: for small systems it is launch-bound (configs[0]: 0.24 ms per
    // step, of which the kernels need a third), so steps 2..n are replayed from a CUDA graph captured on the
    // caller's stream.  Needs a real (capturable) stream and no per-stage timing; step 1 runs plainly so that
    // every kernel attribute is configured outside the capture.
    if (n_steps >= 4 && st != nullptr && !m->timing && n_atoms > 0) {
        nnp_status rc = one_step();
        if (rc != NNP_OK) return rc;
        done = 1;
        DeviceGuard dg(m->device);
        if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
            const int before = launches;
            rc = one_step();
            cudaGraph_t graph = nullptr;
            const cudaError_t ce = cudaStreamEndCapture(st, &graph);
            const int per_step = launches - before;
            launches = before;
            if (rc == NNP_OK && ce == cudaSuccess && graph &&
                cudaGraphInstantiate(&m->md_exec, graph, 0) == cudaSuccess) {
                m->md_exec_stream = st;
                for (; done < n_steps; ++done) {
                    if (cudaGraphLaunch(m->md_exec, st) != cudaSuccess) break;
                    launches += per_step;
                }
            } else {
                cudaGetLastError();     // capture refused: fall back to plain launches below
                m->md_exec = nullptr;
            }
            if (graph) cudaGraphDestroy(graph);
            if (rc != NNP_OK) return rc;
        } else {
            cudaGetLastError();
        }
    }
    for (; done < n_steps; ++done) {
        const nnp_status rc = one_step();
        if (rc != NNP_OK) return rc;
    }
    m->last_launches = launches;
    NNP_CUDA(m, cudaGetLastError());
    return NNP_OK;
}

extern "C" nnp_status nnp_md_kinetic_energy(nnp_model* m, const double* h_mass, int64_t n_atoms, const double* d_vel,
                                            const int32_t* d_type, double* d_ekin, void* d_workspace,
                                            size_t workspace_bytes, void* cuda_stream) {
    if (!m) return NNP_ERR_INVALID_ARG;
    if (!h_mass || !d_ekin || n_atoms < 0 || (n_atoms > 0 && (!d_vel || !d_type))) return fail(m, NNP_ERR_INVALID_ARG, "null array");
    Workspace w;
    const size_t need = ws_layout(&w, d_workspace, n_atoms, m->n_elem, row_stride(m), m->g_stride, skin_stride(m));
    if (!d_workspace || ((uintptr_t)d_workspace & 255u) || workspace_bytes < need)
        return fail(m, NNP_ERR_WORKSPACE, "workspace null, misaligned or too small");
    DeviceGuard dg(m->device);
    if (!dg.ok) return fail(m, NNP_ERR_CUDA, "cudaSetDevice failed");
    launch_ekin(n_atoms, m->n_elem, h_mass, d_type, d_vel, w.partial, d_ekin, (cudaStream_t)cuda_stream);   // the energy partials are scratch between calls
    NNP_CUDA(m, cudaGetLastError());
    return NNP_OK;
}

extern "C" nnp_status nnp_md_kinetic_energy_noalloc(nnp_model* m, const double* h_mass, int64_t n_atoms, const double* d_vel,
                                                    const int32_t* d_type, double* d_ekin, void* cuda_stream) {
    if (!m) return NNP_ERR_INVALID_ARG;
    if (!h_mass || !d_ekin || n_atoms < 0 || (n_atoms > 0 && (!d_vel || !d_type))) return fail(m, NNP_ERR_INVALID_ARG, "null array");
    for (int e = 0; e < m->n_elem; ++e)
        if (!(h_mass[e] > 0.0) || !std::isfinite(h_mass[e])) return fail(m, NNP_ERR_INVALID_ARG, "mass must be finite and > 0");
    if (n_atoms > NOALLOC_MAX_ATOMS)
        return fail(m, NNP_ERR_LIMIT, "n_atoms > NNP_NOALLOC_MAX_ATOMS (4194304): the static scratch array holds 16384 block sums; "
                                      "use nnp_md_kinetic_energy with a workspace");
    DeviceGuard dg(m->device);
    if (!dg.ok) return fail(m, NNP_ERR_CUDA, "cudaSetDevice failed");
    int launches = 0;
    const cudaError_t e = launch_ekin_noalloc(n_atoms, m->n_elem, h_mass, d_type, d_vel, d_ekin, (cudaStream_t)cuda_stream, &launches);
    if (e != cudaSuccess) return fail(m, NNP_ERR_CUDA, std::string("nnp_md_kinetic_energy_noalloc: ") + cudaGetErrorString(e));
    return NNP_OK;
}

extern "C" nnp_status nnp_sync_status(nnp_model* m) {
    if (!m) return NNP_ERR_INVALID_ARG;
    if (!m->have_ws) return NNP_OK;
    DeviceGuard dg(m->device);
    // flags of the last call OR the sticky word (every call since the previous nnp_sync_status: the steps of an
    // nnp_md_run, or several nnp_compute calls enqueued back to back); reading clears the sticky word
    NNP_CUDA(m, cudaMemcpyAsync(m->h_status, m->ws.status, sizeof(int32_t), cudaMemcpyDeviceToHost, m->last_stream));
    NNP_CUDA(m, cudaMemcpyAsync(m->h_status + 1, m->d_sticky, sizeof(int32_t), cudaMemcpyDeviceToHost, m->last_stream));
    NNP_CUDA(m, cudaMemsetAsync(m->d_sticky, 0, sizeof(int32_t), m->last_stream));
    NNP_CUDA(m, cudaStreamSynchronize(m->last_stream));
    const int s = m->h_status[0] | m->h_status[1];
    if (s & ST_NONFINITE) return fail(m, NNP_ERR_NONFINITE, "non-finite position");
    if (s & ST_TYPE_RANGE) return fail(m, NNP_ERR_TYPE_RANGE, "atom type out of range");
    if (s & ST_NBR_OVERFLOW) return fail(m, NNP_ERR_NEIGHBOR_OVERFLOW, "an atom has more than max_neighbors neighbours");
    if (s & ST_FORCE_RANGE) return fail(m, NNP_ERR_FORCE_RANGE, "a force contribution beyond +-2^22 eV/A (deterministic fixed-point accumulation)");
    return NNP_OK;
}

extern "C" nnp_status nnp_compute_host(nnp_model* m, int64_t n, const double* h_pos, const int32_t* h_type,
                                       const double box[3], double* h_e_atom, double* h_e_total, double* h_force) {
    if (!m) return NNP_ERR_INVALID_ARG;
    if (n < 0) return fail(m, NNP_ERR_INVALID_ARG, "n_atoms < 0");
    if (!h_e_total || (n > 0 && (!h_pos || !h_type || !h_e_atom || !h_force))) return fail(m, NNP_ERR_INVALID_ARG, "null array");
    DeviceGuard dg(m->device);
    if (!dg.ok) return fail(m, NNP_ERR_CUDA, "cudaSetDevice failed");
    if (!m->hstream) NNP_CUDA(m, cudaStreamCreateWithFlags(&m->hstream, cudaStreamNonBlocking));
    const size_t need = nnp_workspace_bytes(m, n);
    if (need > m->h_ws_bytes) {
        if (m->h_ws) cudaFree(m->h_ws);
        m->h_ws = nullptr; m->h_ws_bytes = 0;
        NNP_CUDA(m, cudaMalloc(&m->h_ws, need));
        m->h_ws_bytes = need;
    }
    if (n > m->h_cap || !m->hd_etot) {
        if (m->hd_pos) cudaFree(m->hd_pos);
        if (m->hd_type) cudaFree(m->hd_type);
        if (m->hd_e) cudaFree(m->hd_e);
        if (m->hd_f) cudaFree(m->hd_f);
        if (m->hd_etot) cudaFree(m->hd_etot);
        m->hd_pos = m->hd_e = m->hd_f = m->hd_etot = nullptr; m->hd_type = nullptr; m->h_cap = 0;
        const size_t N = (size_t)(n > 0 ? n : 1);
        NNP_CUDA(m, cudaMalloc(&m->hd_pos, N * 24));
        NNP_CUDA(m, cudaMalloc(&m->hd_type, N * 4));
        NNP_CUDA(m, cudaMalloc(&m->hd_e, N * 8));
        NNP_CUDA(m, cudaMalloc(&m->hd_f, N * 24));
        NNP_CUDA(m, cudaMalloc(&m->hd_etot, 8));
        m->h_cap = (int64_t)N;
    }
    if (n > 0) {
        NNP_CUDA(m, cudaMemcpyAsync(m->hd_pos, h_pos, (size_t)n * 24, cudaMemcpyHostToDevice, m->hstream));
        NNP_CUDA(m, cudaMemcpyAsync(m->hd_type, h_type, (size_t)n * 4, cudaMemcpyHostToDevice, m->hstream));
    }
    nnp_status s = nnp_compute(m, n, m->hd_pos, m->hd_type, box, m->hd_e, m->hd_etot, m->hd_f, m->h_ws, m->h_ws_bytes,
                               (void*)m->hstream);
    if (s != NNP_OK) return s;
    if (n > 0) {
        NNP_CUDA(m, cudaMemcpyAsync(h_e_atom, m->hd_e, (size_t)n * 8, cudaMemcpyDeviceToHost, m->hstream));
        NNP_CUDA(m, cudaMemcpyAsync(h_force, m->hd_f, (size_t)n * 24, cudaMemcpyDeviceToHost, m->hstream));
    }
    NNP_CUDA(m, cudaMemcpyAsync(h_e_total, m->hd_etot, 8, cudaMemcpyDeviceToHost, m->hstream));
    return nnp_sync_status(m);
}

// ---------------------------------------------------------------- timing

extern "C" nnp_status nnp_set_timing(nnp_model* m, int32_t enabled) {
    if (!m) return NNP_ERR_INVALID_ARG;
    m->timing = enabled != 0;
    if (!m->timing) m->timing_valid = false;
    return NNP_OK;
}

extern "C" nnp_status nnp_get_timings(nnp_model* m, double* ms) {
    if (!m || !ms) return NNP_ERR_INVALID_ARG;
    if (!m->timing_valid) return fail(m, NNP_ERR_INVALID_ARG, "timing not enabled for the last nnp_compute");
    DeviceGuard dg(m->device);
    NNP_CUDA(m, cudaEventSynchronize(m->ev[NNP_N_STAGES]));
    for (int k = 0; k < NNP_N_STAGES; ++k) {
        float t = 0.f;
        NNP_CUDA(m, cudaEventElapsedTime(&t, m->ev[k], m->ev[k + 1]));
        ms[k] = t;
    }
    return NNP_OK;
}

// ---------------------------------------------------------------- exports

extern "C" nnp_status nnp_get_neighbor_counts(nnp_model* m, int32_t* d_counts) {
    if (!m || !d_counts) return NNP_ERR_INVALID_ARG;
    if (!m->have_ws) return fail(m, NNP_ERR_INVALID_ARG, "no nnp_compute yet");
    DeviceGuard dg(m->device);
    launch_export_counts(m->ws, m->last_n, m->n_elem, d_counts, m->last_stream);
    NNP_CUDA(m, cudaStreamSynchronize(m->last_stream));
    return NNP_OK;
}

extern "C" nnp_status nnp_get_neighbors(nnp_model* m, int64_t* d_offsets, int32_t* d_idx, int64_t idx_capacity) {
    if (!m || !d_offsets) return NNP_ERR_INVALID_ARG;
    if (!m->have_ws) return fail(m, NNP_ERR_INVALID_ARG, "no nnp_compute yet");
    DeviceGuard dg(m->device);
    const int64_t n = m->last_n;
    int32_t* d_counts = nullptr;
    int64_t* d_tmp = nullptr;
    NNP_CUDA(m, cudaMalloc(&d_counts, sizeof(int32_t) * (size_t)(n + 1)));
    cudaError_t e = cudaMalloc(&d_tmp, sizeof(int64_t) * (size_t)(n / 2048 + 16384));
    if (e != cudaSuccess) { cudaFree(d_counts); return fail(m, NNP_ERR_CUDA, cudaGetErrorString(e)); }
    launch_export_counts(m->ws, n, m->n_elem, d_counts, m->last_stream);
    launch_scan_i64_from_i32(d_counts, n, d_offsets, d_tmp, m->last_stream);
    if (d_idx) launch_export_neighbors(m->ws, n, m->n_elem, row_stride(m), d_offsets, d_idx, idx_capacity, m->last_stream);
    e = cudaStreamSynchronize(m->last_stream);
    cudaFree(d_counts);
    cudaFree(d_tmp);
    if (e != cudaSuccess) return fail(m, NNP_ERR_CUDA, cudaGetErrorString(e));
    return NNP_OK;
}

static nnp_status export_rows(nnp_model* m, const double* src, double* dst) {
    if (!m || !dst) return NNP_ERR_INVALID_ARG;
    if (!m->have_ws) return fail(m, NNP_ERR_INVALID_ARG, "no nnp_compute yet");
    DeviceGuard dg(m->device);
    launch_export_rows(m->ws, m->last_n, m->g_stride, src, dst, m->last_stream);
    NNP_CUDA(m, cudaStreamSynchronize(m->last_stream));
    return NNP_OK;
}

extern "C" nnp_status nnp_get_sf(nnp_model* m, double* d_G) { return export_rows(m, m ? m->ws.G : nullptr, d_G); }
extern "C" nnp_status nnp_get_dedg(nnp_model* m, double* d) { return export_rows(m, m ? m->ws.dEdG : nullptr, d); }

extern "C" nnp_status nnp_measure_fp64_peak(int32_t cuda_device, double seconds, double* dfma_per_s,
                                            double* dfma_per_s_sustained) {
    if (!dfma_per_s) return NNP_ERR_INVALID_ARG;
    DeviceGuard dg(cuda_device);
    if (!dg.ok) return NNP_ERR_CUDA;
    cudaError_t e;
    *dfma_per_s = fp64_peak(cuda_device, seconds, dfma_per_s_sustained, &e);
    return e == cudaSuccess ? NNP_OK : NNP_ERR_CUDA;
}

// Host side of libcuhpx.so: argument validation, HEALPix ring geometry, seed / cut-off
// tables, workspace carve-up and the extern "C" entry points of include/cuhpx.h.
//
// The library keeps NO per-workspace state (SURVEY 8(b) "Conventions"): everything a call needs on the host --
// ring lists, cut-offs, launch shapes, table offsets -- is a pure function of (nside, lmax, mmax, batch, dtype)
// and is memoised under that key; device tables are addressed as workspace base + offset, so a workspace may be
// copied, moved or freed by its owner without telling the library.  The first 256 bytes of an initialised
// workspace hold a header (magic, key) that every kernel checks before it trusts a table.
#include <cuda_runtime.h>
#include <math.h>
#include <string.h>

#include <list>
#include <mutex>
#include <vector>

#include "cuhpx_internal.h"

namespace cuhpx {

int legendre_chunk_pairs(cuhpx_dtype_t dt, int batch, int lmax, int npairs);  // legendre.cu
void legendre_start_chunks(cuhpx_dtype_t dt, int npairs, int chunk[2]);            // legendre.cu
cudaError_t launch_legendre_start_tables(const DevPlan& P, cudaStream_t st);         // legendre.cu

namespace {

typedef long double ld;
const ld PI_LD = 3.14159265358979323846264338327950288419716939937510L;

constexpr int MAX_BATCH = 65535;  // channels index gridDim.y / gridDim.z

bool valid_args(int nside, int lmax, int mmax, int batch, int dtype) {
    if (nside < 1 || nside > (1 << 13) || !is_pow2(nside)) return false;
    if (lmax < 0 || mmax < 0 || mmax > lmax || lmax > 4 * (1 << 13)) return false;
    if (batch < 1 || batch > MAX_BATCH) return false;
    if (dtype != CUHPX_F32 && dtype != CUHPX_F64) return false;
    return true;
}

// Which ring grid: HEALPix (n1 = nside) or an iso-latitude grid of n1 rings x n2 equally spaced pixels starting at
// phi = 0 ("generalizes to ... Legendre-Gauss or Lobatto grids").
struct Grid {
    int geometry;  // cuhpx_grid_t
    int n1, n2;
};
constexpr int MAX_NLAT = 1 << 14;

bool valid_grid(const Grid& g) {
    if (g.geometry == CUHPX_GRID_HEALPIX) return g.n1 >= 1 && g.n1 <= (1 << 13) && is_pow2(g.n1) && g.n2 == 0;
    if (g.geometry != CUHPX_GRID_GAUSS_LEGENDRE && g.geometry != CUHPX_GRID_EQUIANGULAR) return false;
    return g.n1 >= 1 && g.n1 <= MAX_NLAT && g.n2 >= 4 && g.n2 <= (1 << 14) && is_pow2(g.n2);
}
int grid_max_ring(const Grid& g) { return g.geometry == CUHPX_GRID_HEALPIX ? 4 * g.n1 : g.n2; }

bool valid_call(const Grid& g, int lmax, int mmax, int batch, int dtype) {
    if (!valid_grid(g)) return false;
    if (g.geometry == CUHPX_GRID_HEALPIX) return valid_args(g.n1, lmax, mmax, batch, dtype);
    if (lmax < 0 || mmax < 0 || mmax > lmax || lmax > 4 * (1 << 13)) return false;
    if (batch < 1 || batch > MAX_BATCH) return false;
    return dtype == CUHPX_F32 || dtype == CUHPX_F64;
}

// Gorski et al. ring table, northern hemisphere incl. equator: ring pair j (0-based) <-> ring i = j + 1.
struct PairGeom {
    int N;
    long long start;
    int shifted;
    ld y;    // 1 - cos(theta), exact rational rounded once
    ld sth;  // sin(theta)
    ld w;    // quadrature weight per pixel (iso-latitude grids)
};

// Gauss-Legendre nodes (as colatitudes, north first) and weights by Newton's iteration on P_n(cos theta) in the angle,
// long double; weights sum to 2.  (Textbook: Abramowitz & Stegun 25.4.29; the three-term recurrence for P_n.)
void gauss_legendre(int n, std::vector<ld>& theta, std::vector<ld>& w) {
    theta.resize(n);
    w.resize(n);
    for (int k = 0; k < (n + 1) / 2; ++k) {
        ld t = PI_LD * ((ld)k + 0.75L) / ((ld)n + 0.5L);  // Tricomi's initial guess
        ld dp = 0;
        for (int it = 0; it < 100; ++it) {
            const ld x = cosl(t);
            ld p0 = 1, p1 = x;
            for (int l = 2; l <= n; ++l) {
                const ld p2 = ((2 * l - 1) * x * p1 - (l - 1) * p0) / l;
                p0 = p1;
                p1 = p2;
            }
            if (n == 1) { p0 = 1; p1 = x; }
            dp = n * (x * p1 - p0) / (x * x - 1);      // dP_n/dx
            const ld dt = p1 / (dp * -sinl(t));        // Newton in theta: d/dtheta = -sin(theta) d/dx
            t -= dt;
            if (fabsl(dt) < 1e-19L) break;
        }
        const ld x = cosl(t);
        ld p0 = 1, p1 = x;
        for (int l = 2; l <= n; ++l) {
            const ld p2 = ((2 * l - 1) * x * p1 - (l - 1) * p0) / l;
            p0 = p1;
            p1 = p2;
        }
        dp = n * (x * p1 - p0) / (x * x - 1);
        theta[k] = t;
        theta[n - 1 - k] = PI_LD - t;
        w[k] = w[n - 1 - k] = 2 / ((1 - x * x) * dp * dp);
    }
}

// Fejer's first rule on theta_k = pi (k + 1/2) / n: exact for polynomials in cos(theta) of degree <= n - 1; weights sum to 2
void fejer1(int n, std::vector<ld>& theta, std::vector<ld>& w) {
    theta.resize(n);
    w.resize(n);
    for (int k = 0; k < n; ++k) {
        const ld t = PI_LD * ((ld)k + 0.5L) / (ld)n;
        ld s = 0;
        for (int j = 1; j <= n / 2; ++j) s += cosl(2 * j * t) / (ld)(4LL * j * j - 1);
        theta[k] = t;
        w[k] = 2 * (1 - 2 * s) / (ld)n;
    }
}

PairGeom pair_geom(int nside, int j) {
    PairGeom g;
    g.w = 0;
    const long long ns = nside, i = j + 1;
    if (i < ns) {  // polar cap: N = 4 i, z = 1 - i^2 / (3 nside^2), phi0 = pi / N
        g.N = (int)(4 * i);
        g.start = 2 * i * (i - 1);
        g.shifted = 1;
        g.y = (ld)(i * i) / (ld)(3 * ns * ns);
    } else {  // belt: N = 4 nside, z = 4/3 - 2 i / (3 nside), shifted when (i - nside) is even
        g.N = (int)(4 * ns);
        g.start = 2 * ns * (ns - 1) + (i - ns) * 4 * ns;
        g.shifted = ((i - ns) % 2 == 0) ? 1 : 0;
        g.y = (ld)(2 * i - ns) / (ld)(3 * ns);
    }
    g.sth = sqrtl(g.y * (2.0L - g.y));
    return g;
}

inline void split_hi_lo(ld v, double& hi, double& lo) {
    hi = (double)v;
    lo = (double)(v - (ld)hi);
}

size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

// Does ring pair j take part at order m, i.e. does |lambda_lm(theta_j)| reach 2^-110 for some l <= lmax?
// (Scaled fp64 recurrence; the device kernels use the same criterion only through the tables built here.)
bool pair_active(int lmax, int m, ld pref_m, ld lg2sin, double yj) {
    const double NEG = -110.0;
    ld e = pref_m + (ld)m * lg2sin;  // log2 |lambda_mm|
    if (e >= NEG) return true;
    double ex = (double)e;
    double cur = 1.0, prev = 0.0;
    const double dm = (double)m;
    for (int l = m + 1; l <= lmax; ++l) {
        const double dl = (double)l;
        const double l2m2 = (dl - dm) * (dl + dm);
        const double A = sqrt((4.0 * dl * dl - 1.0) / l2m2);
        const double num = (2.0 * dl + 1.0) * ((dl - 1.0 - dm) * (dl - 1.0 + dm));
        const double B = num == 0.0 ? 0.0 : -sqrt(num / ((2.0 * dl - 3.0) * l2m2));
        const double nx = A * (cur - yj * cur) + B * prev;
        prev = cur;
        cur = nx;
        const double ac = fabs(cur);
        if (ac > 0x1p300) {
            cur *= 0x1p-300;
            prev *= 0x1p-300;
            ex += 300.0;
        }
        if (ac > 0.0 && ex + (double)ilogb(cur) >= NEG) return true;
        // once lambda stops growing (past the turning point) it never will again
        if (l > m + 2 && fabs(cur) < fabs(prev) && ex + (double)ilogb(prev) < NEG - 60) return false;
    }
    return false;
}

// Everything the host needs for (nside, lmax, mmax, batch, dtype): geometry, seeds, cut-offs, FFT ring classes, offsets.
HostPlan* make_plan(const Grid& grid, int lmax, int mmax, int batch, cuhpx_dtype_t dt) {
    HostPlan* hp = new HostPlan;
    DevPlan& d = hp->d;
    memset(&d, 0, sizeof(d));
    hp->dtype = dt;
    hp->geometry = grid.geometry;
    const bool hpx = grid.geometry == CUHPX_GRID_HEALPIX;
    const int nside = hpx ? grid.n1 : 0;
    d.nside = nside;
    d.lmax = lmax;
    d.mmax = mmax;
    d.batch = batch;
    d.nrings = hpx ? 4 * nside - 1 : grid.n1;
    d.npairs = hpx ? 2 * nside : (grid.n1 + 1) / 2;
    d.mstride = (int)cuhpx_spectra_stride(mmax);
    d.npix = hpx ? 12LL * nside * nside : (long long)grid.n1 * grid.n2;
    d.nalm = (long long)cuhpx_alm_count(lmax, mmax);
    d.key = plan_key(grid.n1, lmax, mmax, batch, (int)dt, grid.geometry + 16 * grid.n2);
    hp->max_ring = grid_max_ring(grid);
    std::vector<ld> gtheta, gw;
    if (grid.geometry == CUHPX_GRID_GAUSS_LEGENDRE) gauss_legendre(grid.n1, gtheta, gw);
    if (grid.geometry == CUHPX_GRID_EQUIANGULAR) fejer1(grid.n1, gtheta, gw);
    if (!hpx) {  // quadrature weight per pixel: w_ring * 2 pi / nlon (Eq. 26 with the grid's own W)
        hp->h_weight.resize(d.nrings);
        for (int r = 0; r < d.nrings; ++r) hp->h_weight[r] = (double)(gw[r] * 2 * PI_LD / (ld)grid.n2);
    }
    d.chunk_pairs = legendre_chunk_pairs(dt, batch, lmax, d.npairs);
    d.nchunk_max = (d.npairs + d.chunk_pairs - 1) / d.chunk_pairs;

    // ---- per-pair and per-m tables (long double on the host)
    hp->h_ringN.resize(d.npairs);
    hp->h_start.resize(d.npairs);
    hp->h_shifted.resize(d.npairs);
    hp->h_y.resize(d.npairs);
    hp->h_lshi.resize(d.npairs);
    hp->h_lslo.resize(d.npairs);
    hp->h_prefhi.resize(mmax + 1);
    hp->h_preflo.resize(mmax + 1);
    std::vector<ld> lg2sin(d.npairs), pref(mmax + 1);
    for (int j = 0; j < d.npairs; ++j) {
        PairGeom g;
        if (hpx) {
            g = pair_geom(nside, j);
        } else {  // ring j of the northern half (the middle ring of an odd count is its own mirror)
            g.N = grid.n2;
            g.start = (long long)j * grid.n2;
            g.shifted = 0;
            const ld h = sinl(gtheta[j] / 2);
            g.y = 2 * h * h;  // 1 - cos(theta) without cancellation
            g.sth = sinl(gtheta[j]);
            g.w = gw[j];
        }
        hp->h_ringN[j] = g.N;
        hp->h_start[j] = g.start;
        hp->h_shifted[j] = g.shifted;
        hp->h_y[j] = (double)g.y;
        lg2sin[j] = log2l(g.sth);
        split_hi_lo(lg2sin[j], hp->h_lshi[j], hp->h_lslo[j]);
    }
    // log2 |lambda_mm| = -0.5 log2(4 pi) + 0.5 sum_{k<=m} log2(1 + 1/(2k)) + m log2 sin(theta)   (Eq. 15)
    ld acc = -0.5L * log2l(4.0L * PI_LD);
    for (int m = 0; m <= mmax; ++m) {
        if (m > 0) acc += 0.5L * log1pl(1.0L / (2.0L * m)) / logl(2.0L);
        pref[m] = acc;
        split_hi_lo(acc, hp->h_prefhi[m], hp->h_preflo[m]);
    }
    // ---- jmin[m]: first ring pair that matters at order m (two-pointer: the active set shrinks with m)
    hp->h_jmin.assign(mmax + 1, 0);
    int j = 0;
    for (int m = 0; m <= mmax; ++m) {
        while (j < d.npairs - 1 && !pair_active(lmax, m, pref[m], lg2sin[j], hp->h_y[j])) ++j;
        hp->h_jmin[m] = j;
    }
    // ---- mcut[j]: last order at which pair j is processed (monotone non-decreasing in j, as the sweep implies)
    hp->h_mcut.assign(d.npairs, 0);
    {
        int m = mmax;
        for (int jj = d.npairs - 1; jj >= 0; --jj) {
            while (m > 0 && hp->h_jmin[m] > jj) --m;
            hp->h_mcut[jj] = m;
        }
    }

    // ---- workspace layout
    size_t o = 256;  // header
    auto take = [&](size_t bytes) {
        size_t r = o;
        o = align_up(o + bytes);
        return r;
    };
    hp->off_y = take(sizeof(double) * d.npairs);
    hp->off_lshi = take(sizeof(double) * d.npairs);
    hp->off_lslo = take(sizeof(double) * d.npairs);
    hp->off_ringN = take(sizeof(int) * d.npairs);
    hp->off_start = take(sizeof(long long) * d.npairs);
    hp->off_shifted = take(sizeof(int) * d.npairs);
    hp->off_mcut = take(sizeof(int) * d.npairs);
    hp->off_prefhi = take(sizeof(double) * (d.mmax + 1));
    hp->off_preflo = take(sizeof(double) * (d.mmax + 1));
    hp->off_jmin = take(sizeof(int) * (d.mmax + 1));
    hp->off_defw = hpx ? 0 : take(sizeof(double) * d.nrings);
    hp->off_fft = o;
    hp->fft_bytes = fft_plan_host(*hp);
    o = align_up(o + hp->fft_bytes);
    hp->off_alpha = take(sizeof(double) * (size_t)d.nalm);
    hp->off_scale = take(sizeof(double) * (size_t)d.nalm);
    const size_t csize = dt == CUHPX_F64 ? 16 : 8;
    hp->off_spectra = take(csize * (size_t)d.batch * d.nrings * d.mstride);
    hp->off_partial = o;
    if (d.nchunk_max > 1) take(csize * (size_t)d.nchunk_max * d.batch * d.nalm);
    // tensor-core Legendre path: per-call operand images (stages of 32 degrees, see legendre_tc.cu)
    d.tc_nb = legendre_tc_group(dt, batch);
    hp->off_tcprefix = hp->off_tcimages = 0;
    if (d.tc_nb > 0) {
        hp->h_tcprefix.assign(mmax + 2, 0);
        for (int m = 0; m <= mmax; ++m) hp->h_tcprefix[m + 1] = hp->h_tcprefix[m] + (lmax - m + 1 + 31) / 32;
        hp->off_tcprefix = take(sizeof(long long) * (mmax + 2));
        const size_t groups = (size_t)(batch + d.tc_nb - 1) / d.tc_nb;
        hp->off_tcimages = take(groups * (size_t)hp->h_tcprefix[mmax + 1] * legendre_tc_image_bytes(d.tc_nb));
    }
    // late-start tables of the fp64 Legendre kernels (legendre.cu)
    legendre_start_chunks(dt, d.npairs, d.st_chunk);
    for (int k = 0; k < 2; ++k) {
        d.st_nchunk[k] = 0;
        if (d.st_chunk[k] <= 0) continue;
        d.st_nchunk[k] = (d.npairs + d.st_chunk[k] - 1) / d.st_chunk[k];
        const size_t n = (size_t)(mmax + 1) * d.npairs;
        hp->off_st[k][0] = take(sizeof(double) * n);
        hp->off_st[k][1] = take(sizeof(double) * n);
        hp->off_st[k][2] = take(sizeof(int) * n);
        hp->off_st[k][3] = take(sizeof(int) * (size_t)(mmax + 1) * d.st_nchunk[k]);
    }
    hp->workspace_bytes = o;
    return hp;
}

// memo of host plans (bounded; entries are immutable and shared, so eviction never invalidates a running call)
struct PlanKey {
    int geometry, n1, n2, lmax, mmax, batch, dtype;
    bool operator==(const PlanKey& o) const {
        return geometry == o.geometry && n1 == o.n1 && n2 == o.n2 && lmax == o.lmax && mmax == o.mmax && batch == o.batch &&
               dtype == o.dtype;
    }
};
std::mutex g_mu;
std::list<std::pair<PlanKey, PlanRef>> g_plans;  // most recently used first
constexpr size_t MAX_PLANS = 24;

PlanRef get_plan(const Grid& grid, int lmax, int mmax, int batch, cuhpx_dtype_t dt);
PlanRef get_plan(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dt) {
    return get_plan(Grid{CUHPX_GRID_HEALPIX, nside, 0}, lmax, mmax, batch, dt);
}
PlanRef get_plan(const Grid& grid, int lmax, int mmax, int batch, cuhpx_dtype_t dt) {
    const PlanKey k{grid.geometry, grid.n1, grid.n2, lmax, mmax, batch, (int)dt};
    {
        std::lock_guard<std::mutex> lk(g_mu);
        for (auto it = g_plans.begin(); it != g_plans.end(); ++it)
            if (it->first == k) {
                g_plans.splice(g_plans.begin(), g_plans, it);
                return g_plans.front().second;
            }
    }
    PlanRef p(make_plan(grid, lmax, mmax, batch, dt));  // built outside the lock (may take a while at nside 4096)
    std::lock_guard<std::mutex> lk(g_mu);
    for (auto& e : g_plans)
        if (e.first == k) return e.second;
    g_plans.emplace_front(k, p);
    while (g_plans.size() > MAX_PLANS) g_plans.pop_back();
    return p;
}

bool overlap(const void* a, size_t na, const void* b, size_t nb) {
    const uintptr_t pa = (uintptr_t)a, pb = (uintptr_t)b;
    return pa < pb + nb && pb < pa + na;
}

size_t map_bytes(const HostPlan& hp) { return (size_t)hp.d.batch * (size_t)hp.d.npix * (hp.dtype == CUHPX_F64 ? 8 : 4); }
size_t alm_bytes(const HostPlan& hp) { return (size_t)hp.d.batch * (size_t)hp.d.nalm * (hp.dtype == CUHPX_F64 ? 16 : 8); }

// Argument checks shared by the operators; a / b are the data buffers with their sizes (either may be null for the
// stage-level calls, which touch only one user buffer).
int check_call(PlanRef* out, const Grid& grid, int lmax, int mmax, int batch, int dt, const void* a, size_t na, const void* b,
               size_t nb, const void* ws, size_t ws_bytes);
int check_call(PlanRef* out, int nside, int lmax, int mmax, int batch, int dt, const void* a, size_t na, const void* b,
               size_t nb, const void* ws, size_t ws_bytes) {
    return check_call(out, Grid{CUHPX_GRID_HEALPIX, nside, 0}, lmax, mmax, batch, dt, a, na, b, nb, ws, ws_bytes);
}
int check_call(PlanRef* out, const Grid& grid, int lmax, int mmax, int batch, int dt, const void* a, size_t na, const void* b,
               size_t nb, const void* ws, size_t ws_bytes) {
    if (!valid_call(grid, lmax, mmax, batch, dt)) return CUHPX_EINVAL;
    if ((na && !a) || (nb && !b) || !ws) return CUHPX_EINVAL;
    if (((uintptr_t)a & 15) || ((uintptr_t)b & 15) || ((uintptr_t)ws & 15)) return CUHPX_EINVAL;
    // the map may hold up to 4 nside * 4 nside-ish rings of any supported length; unsupported ring lengths were
    // refused by cuhpx_workspace_bytes / cuhpx_workspace_init already
    if (!fft_supported(grid_max_ring(grid), (cuhpx_dtype_t)dt)) return CUHPX_EUNSUPPORTED;
    PlanRef hp = get_plan(grid, lmax, mmax, batch, (cuhpx_dtype_t)dt);
    if (ws_bytes < hp->workspace_bytes) return CUHPX_EWORKSPACE;
    const size_t sa = a ? (na == (size_t)-1 ? map_bytes(*hp) : na == (size_t)-2 ? alm_bytes(*hp) : na) : 0;
    const size_t sb = b ? (nb == (size_t)-1 ? map_bytes(*hp) : nb == (size_t)-2 ? alm_bytes(*hp) : nb) : 0;
    if (a && b && overlap(a, sa, b, sb)) return CUHPX_EINVAL;
    if (a && overlap(a, sa, ws, hp->workspace_bytes)) return CUHPX_EINVAL;
    if (b && overlap(b, sb, ws, hp->workspace_bytes)) return CUHPX_EINVAL;
    *out = hp;
    return CUHPX_OK;
}
constexpr size_t MAP = (size_t)-1, ALM = (size_t)-2;  // "size of one map / alm array of this plan"

}  // namespace

DevPlan HostPlan::resolve(void* ws) const {
    DevPlan P = d;
    char* base = (char*)ws;
    P.hdr = (const WsHeader*)base;
    P.y = (const double*)(base + off_y);
    P.ls_hi = (const double*)(base + off_lshi);
    P.ls_lo = (const double*)(base + off_lslo);
    P.ringN = (const int*)(base + off_ringN);
    P.start = (const long long*)(base + off_start);
    P.shifted = (const int*)(base + off_shifted);
    P.mcut = (const int*)(base + off_mcut);
    P.pref_hi = (const double*)(base + off_prefhi);
    P.pref_lo = (const double*)(base + off_preflo);
    P.jmin = (const int*)(base + off_jmin);
    P.defw = off_defw ? (const double*)(base + off_defw) : nullptr;
    P.coef_alpha = (const double*)(base + off_alpha);
    P.coef_scale = (const double*)(base + off_scale);
    P.spectra = base + off_spectra;
    P.partial = d.nchunk_max > 1 ? base + off_partial : nullptr;
    P.tc_prefix = d.tc_nb > 0 ? (const long long*)(base + off_tcprefix) : nullptr;
    P.tc_images = d.tc_nb > 0 ? base + off_tcimages : nullptr;
    for (int k = 0; k < 2; ++k) {
        const bool on = d.st_chunk[k] > 0;
        P.st_cur[k] = on ? (const double*)(base + off_st[k][0]) : nullptr;
        P.st_prev[k] = on ? (const double*)(base + off_st[k][1]) : nullptr;
        P.st_sc[k] = on ? (const int*)(base + off_st[k][2]) : nullptr;
        P.st_l0[k] = on ? (const int*)(base + off_st[k][3]) : nullptr;
    }
    return P;
}

}  // namespace cuhpx

using namespace cuhpx;

extern "C" {

size_t cuhpx_npix(int nside) {
    if (nside < 1 || !is_pow2(nside)) return 0;
    return (size_t)12 * nside * nside;
}

size_t cuhpx_nrings(int nside) {
    if (nside < 1 || !is_pow2(nside)) return 0;
    return (size_t)4 * nside - 1;
}

size_t cuhpx_alm_count(int lmax, int mmax) {
    if (lmax < 0 || mmax < 0 || mmax > lmax) return 0;
    return (size_t)(mmax + 1) * (lmax + 1) - (size_t)mmax * (mmax + 1) / 2;
}

size_t cuhpx_alm_index(int lmax, int l, int m) { return (size_t)m * (2 * (size_t)lmax + 1 - m) / 2 + l; }

size_t cuhpx_spectra_stride(int mmax) { return (size_t)((mmax + 1 + 1) / 2 * 2); }

const char* cuhpx_status_string(int s) {
    switch (s) {
        case CUHPX_OK: return "CUHPX_OK";
        case CUHPX_EINVAL: return "CUHPX_EINVAL: bad nside/lmax/mmax/batch/dtype or null/misaligned/overlapping pointer";
        case CUHPX_EWORKSPACE: return "CUHPX_EWORKSPACE: workspace too small, not initialised or for other parameters";
        case CUHPX_EUNSUPPORTED: return "CUHPX_EUNSUPPORTED: request not supported by this build";
        case CUHPX_ECUDA: return "CUHPX_ECUDA: CUDA runtime error (see cudaGetLastError)";
    }
    return "unknown status";
}

int cuhpx_ring_info(int nside, int ring, long long* n_pix, long long* first_pix, double* cos_theta, double* phi0) {
    if (nside < 1 || !is_pow2(nside) || ring < 1 || ring > 4 * nside - 1) return CUHPX_EINVAL;
    const int nrings = 4 * nside - 1;
    const int r0 = ring - 1;
    const int j = r0 < nrings - 1 - r0 ? r0 : nrings - 1 - r0;
    PairGeom g = pair_geom(nside, j);
    const bool south = r0 > j;
    if (n_pix) *n_pix = g.N;
    if (first_pix) *first_pix = south ? 12LL * nside * nside - g.N - g.start : g.start;
    if (cos_theta) *cos_theta = (double)(south ? -(1.0L - g.y) : (1.0L - g.y));
    if (phi0) *phi0 = g.shifted ? (double)(PI_LD / (ld)g.N) : 0.0;
    return CUHPX_OK;
}

size_t cuhpx_workspace_bytes(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype) {
    if (!valid_args(nside, lmax, mmax, batch, dtype) || !fft_supported(4 * nside, dtype)) return 0;
    return get_plan(nside, lmax, mmax, batch, dtype)->workspace_bytes;
}

static int workspace_init_impl(const Grid& grid, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, void* ws, size_t ws_bytes,
                               cuhpx_stream_t stream) {
    if (!valid_call(grid, lmax, mmax, batch, dtype)) return CUHPX_EINVAL;
    if (!ws || ((uintptr_t)ws & 15)) return CUHPX_EINVAL;
    if (!fft_supported(grid_max_ring(grid), dtype)) return CUHPX_EUNSUPPORTED;
    const int nside = grid.n1;
    PlanRef hp = get_plan(grid, lmax, mmax, batch, dtype);
    if (ws_bytes < hp->workspace_bytes) return CUHPX_EWORKSPACE;
    const DevPlan& d = hp->d;
    char* base = (char*)ws;
    cudaStream_t st = (cudaStream_t)stream;

    cudaError_t e = cudaSuccess;
    auto up = [&](size_t off, const void* src, size_t bytes) {
        if (e == cudaSuccess) e = cudaMemcpyAsync(base + off, src, bytes, cudaMemcpyHostToDevice, st);
    };
    // a header that matches nothing while the tables are being (re)built
    WsHeader hdr;
    memset(&hdr, 0, sizeof(hdr));
    up(0, &hdr, sizeof(hdr));
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);  // hdr is rewritten below; the copy must have read it
    up(hp->off_y, hp->h_y.data(), sizeof(double) * d.npairs);
    up(hp->off_lshi, hp->h_lshi.data(), sizeof(double) * d.npairs);
    up(hp->off_lslo, hp->h_lslo.data(), sizeof(double) * d.npairs);
    up(hp->off_ringN, hp->h_ringN.data(), sizeof(int) * d.npairs);
    up(hp->off_start, hp->h_start.data(), sizeof(long long) * d.npairs);
    up(hp->off_shifted, hp->h_shifted.data(), sizeof(int) * d.npairs);
    up(hp->off_mcut, hp->h_mcut.data(), sizeof(int) * d.npairs);
    up(hp->off_prefhi, hp->h_prefhi.data(), sizeof(double) * (mmax + 1));
    up(hp->off_preflo, hp->h_preflo.data(), sizeof(double) * (mmax + 1));
    up(hp->off_jmin, hp->h_jmin.data(), sizeof(int) * (mmax + 1));
    if (hp->off_defw) up(hp->off_defw, hp->h_weight.data(), sizeof(double) * d.nrings);
    if (d.tc_nb > 0) up(hp->off_tcprefix, hp->h_tcprefix.data(), sizeof(long long) * (mmax + 2));
    if (e == cudaSuccess)
        e = launch_legendre_coeff(lmax, mmax, (double*)(base + hp->off_alpha), (double*)(base + hp->off_scale), st);
    if (e == cudaSuccess) e = fft_build_tables(*hp, base + hp->off_fft, st);
    if (e == cudaSuccess) e = launch_legendre_start_tables(hp->resolve(ws), st);
    hdr.magic = WS_MAGIC;
    hdr.key = d.key;
    hdr.nside = nside;
    hdr.lmax = lmax;
    hdr.mmax = mmax;
    hdr.batch = batch;
    hdr.dtype = (int)dtype;
    hdr.geometry = hp->geometry;
    hdr.bytes = hp->workspace_bytes;
    up(0, &hdr, sizeof(hdr));
    // the sources above are pageable host memory owned by the (shared, immutable) plan or by this frame
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    return e == cudaSuccess ? CUHPX_OK : CUHPX_ECUDA;
}

int cuhpx_workspace_init(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, void* ws, size_t ws_bytes,
                         cuhpx_stream_t stream) {
    return workspace_init_impl(Grid{CUHPX_GRID_HEALPIX, nside, 0}, lmax, mmax, batch, dtype, ws, ws_bytes, stream);
}

int cuhpx_workspace_check(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, const void* ws, size_t ws_bytes,
                          cuhpx_stream_t stream) {
    if (!valid_args(nside, lmax, mmax, batch, dtype)) return CUHPX_EINVAL;
    if (!ws || ((uintptr_t)ws & 15)) return CUHPX_EINVAL;
    if (!fft_supported(4 * nside, dtype)) return CUHPX_EUNSUPPORTED;
    PlanRef hp = get_plan(nside, lmax, mmax, batch, dtype);
    if (ws_bytes < hp->workspace_bytes) return CUHPX_EWORKSPACE;
    WsHeader hdr;
    if (cudaMemcpyAsync(&hdr, ws, sizeof(hdr), cudaMemcpyDeviceToHost, (cudaStream_t)stream) != cudaSuccess) return CUHPX_ECUDA;
    if (cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess) return CUHPX_ECUDA;
    if (hdr.magic != WS_MAGIC || hdr.key != hp->d.key || hdr.bytes != hp->workspace_bytes || hdr.bad) return CUHPX_EWORKSPACE;
    return CUHPX_OK;
}

size_t cuhpx_spectra_offset(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype) {
    if (!valid_args(nside, lmax, mmax, batch, dtype) || !fft_supported(4 * nside, dtype)) return 0;
    return get_plan(nside, lmax, mmax, batch, dtype)->off_spectra;
}

int cuhpx_plan_mcut(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, int* h_mcut) {
    if (!valid_args(nside, lmax, mmax, batch, dtype) || !h_mcut) return CUHPX_EINVAL;
    if (!fft_supported(4 * nside, dtype)) return CUHPX_EUNSUPPORTED;
    PlanRef hp = get_plan(nside, lmax, mmax, batch, dtype);
    const DevPlan& d = hp->d;
    for (int r = 0; r < d.nrings; ++r) {
        const int j = r < d.nrings - 1 - r ? r : d.nrings - 1 - r;
        h_mcut[r] = hp->h_mcut[j];
    }
    return CUHPX_OK;
}

int cuhpx_plan_stats(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, double* out, int count) {
    if (!valid_args(nside, lmax, mmax, batch, dtype) || !out || count < 1) return CUHPX_EINVAL;
    if (!fft_supported(4 * nside, dtype)) return CUHPX_EUNSUPPORTED;
    PlanRef hp = get_plan(nside, lmax, mmax, batch, dtype);
    const DevPlan& d = hp->d;
    double st[8] = {0};
    int fl = 0;
    double tb = 0;
    fft_stage_stats(*hp, &fl, &tb);
    st[0] = fl;
    st[1] = d.nchunk_max > 1 ? 2 : 1;
    st[2] = d.tc_nb > 0 ? 2 : 1;  // tensor-core synthesis: operand images + main kernel
    for (int m = 0; m <= d.mmax; ++m) st[3] += (double)(d.lmax - m + 1) * (double)(d.npairs - hp->h_jmin[m]);
    st[4] = (double)d.nalm * (double)d.npairs;
    for (int r = 0; r < d.nrings; ++r) st[5] += hp->h_mcut[r < d.nrings - 1 - r ? r : d.nrings - 1 - r] + 1;
    st[6] = tb;
    st[7] = (double)hp->workspace_bytes;
    for (int i = 0; i < count && i < 8; ++i) out[i] = st[i];
    return CUHPX_OK;
}

int cuhpx_late_start_stats(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, const void* ws, size_t ws_bytes,
                           cuhpx_stream_t stream, double* h_skipped) {
    if (!valid_args(nside, lmax, mmax, batch, dtype) || !ws || ((uintptr_t)ws & 15) || !h_skipped) return CUHPX_EINVAL;
    const int rc = cuhpx_workspace_check(nside, lmax, mmax, batch, dtype, ws, ws_bytes, stream);
    if (rc != CUHPX_OK) return rc;
    PlanRef hp = get_plan(nside, lmax, mmax, batch, dtype);
    const DevPlan& d = hp->d;
    for (int k = 0; k < 2; ++k) {
        h_skipped[k] = 0.0;
        if (d.st_chunk[k] <= 0) continue;
        std::vector<int> l0((size_t)(mmax + 1) * d.st_nchunk[k]);
        if (cudaMemcpyAsync(l0.data(), (const char*)ws + hp->off_st[k][3], sizeof(int) * l0.size(), cudaMemcpyDeviceToHost,
                            (cudaStream_t)stream) != cudaSuccess ||
            cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess)
            return CUHPX_ECUDA;
        for (int m = 0; m <= mmax; ++m)
            for (int c = 0; c < d.st_nchunk[k]; ++c) {
                const long long left = (long long)d.npairs - (hp->h_jmin[m] + (long long)c * d.st_chunk[k]);
                const long long pairs = left < 0 ? 0 : left < d.st_chunk[k] ? left : d.st_chunk[k];
                h_skipped[k] += (double)l0[(size_t)m * d.st_nchunk[k] + c] * (double)pairs;
            }
    }
    return CUHPX_OK;
}

#define CUDA_OR_FAIL(expr)                         \
    do {                                           \
        if ((expr) != cudaSuccess) return CUHPX_ECUDA; \
    } while (0)

int cuhpx_analysis_fft_stage(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dt, const void* d_map,
                             const double* d_w, int use_w, void* ws, size_t ws_bytes, cuhpx_stream_t stream) {
    PlanRef hp;
    int rc = check_call(&hp, nside, lmax, mmax, batch, dt, d_map, MAP, nullptr, 0, ws, ws_bytes);
    if (rc) return rc;
    if (d_w && ((uintptr_t)d_w & 7)) return CUHPX_EINVAL;
    CUDA_OR_FAIL(launch_fft_analysis(*hp, hp->resolve(ws), d_map, d_w, use_w, (cudaStream_t)stream));
    return CUHPX_OK;
}

int cuhpx_analysis_legendre_stage(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dt, void* d_alm, int adjoint,
                                  void* ws, size_t ws_bytes, cuhpx_stream_t stream) {
    PlanRef hp;
    int rc = check_call(&hp, nside, lmax, mmax, batch, dt, d_alm, ALM, nullptr, 0, ws, ws_bytes);
    if (rc) return rc;
    CUDA_OR_FAIL(launch_legendre_analysis(*hp, hp->resolve(ws), d_alm, adjoint, (cudaStream_t)stream));
    return CUHPX_OK;
}

int cuhpx_synthesis_legendre_stage(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dt, const void* d_alm,
                                   int adjoint, void* ws, size_t ws_bytes, cuhpx_stream_t stream) {
    PlanRef hp;
    int rc = check_call(&hp, nside, lmax, mmax, batch, dt, d_alm, ALM, nullptr, 0, ws, ws_bytes);
    if (rc) return rc;
    CUDA_OR_FAIL(launch_legendre_synthesis(*hp, hp->resolve(ws), d_alm, adjoint, (cudaStream_t)stream));
    return CUHPX_OK;
}

int cuhpx_synthesis_fft_stage(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dt, void* d_map, const double* d_w,
                              int use_w, void* ws, size_t ws_bytes, cuhpx_stream_t stream) {
    PlanRef hp;
    int rc = check_call(&hp, nside, lmax, mmax, batch, dt, d_map, MAP, nullptr, 0, ws, ws_bytes);
    if (rc) return rc;
    if (d_w && ((uintptr_t)d_w & 7)) return CUHPX_EINVAL;
    CUDA_OR_FAIL(launch_fft_synthesis(*hp, hp->resolve(ws), d_map, d_w, use_w, (cudaStream_t)stream));
    return CUHPX_OK;
}

int cuhpx_map2alm(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dt, const void* d_map, void* d_alm,
                  const double* d_w, void* ws, size_t ws_bytes, cuhpx_stream_t stream) {
    PlanRef hp;
    int rc = check_call(&hp, nside, lmax, mmax, batch, dt, d_map, MAP, d_alm, ALM, ws, ws_bytes);
    if (rc) return rc;
    if (d_w && ((uintptr_t)d_w & 7)) return CUHPX_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const DevPlan P = hp->resolve(ws);
    CUDA_OR_FAIL(launch_fft_analysis(*hp, P, d_map, d_w, 1, st));
    CUDA_OR_FAIL(launch_legendre_analysis(*hp, P, d_alm, 0, st));
    return CUHPX_OK;
}

int cuhpx_alm2map_adjoint(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dt, const void* d_gmap,
                          void* d_galm, void* ws, size_t ws_bytes, cuhpx_stream_t stream) {
    PlanRef hp;
    int rc = check_call(&hp, nside, lmax, mmax, batch, dt, d_gmap, MAP, d_galm, ALM, ws, ws_bytes);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const DevPlan P = hp->resolve(ws);
    CUDA_OR_FAIL(launch_fft_analysis(*hp, P, d_gmap, nullptr, 0, st));
    CUDA_OR_FAIL(launch_legendre_analysis(*hp, P, d_galm, 1, st));
    return CUHPX_OK;
}

int cuhpx_alm2map(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dt, const void* d_alm, void* d_map,
                  void* ws, size_t ws_bytes, cuhpx_stream_t stream) {
    PlanRef hp;
    int rc = check_call(&hp, nside, lmax, mmax, batch, dt, d_alm, ALM, d_map, MAP, ws, ws_bytes);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const DevPlan P = hp->resolve(ws);
    CUDA_OR_FAIL(launch_legendre_synthesis(*hp, P, d_alm, 0, st));
    CUDA_OR_FAIL(launch_fft_synthesis(*hp, P, d_map, nullptr, 0, st));
    return CUHPX_OK;
}

int cuhpx_map2alm_adjoint(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dt, const void* d_galm,
                          void* d_gmap, const double* d_w, void* ws, size_t ws_bytes, cuhpx_stream_t stream) {
    PlanRef hp;
    int rc = check_call(&hp, nside, lmax, mmax, batch, dt, d_galm, ALM, d_gmap, MAP, ws, ws_bytes);
    if (rc) return rc;
    if (d_w && ((uintptr_t)d_w & 7)) return CUHPX_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const DevPlan P = hp->resolve(ws);
    CUDA_OR_FAIL(launch_legendre_synthesis(*hp, P, d_galm, 1, st));
    CUDA_OR_FAIL(launch_fft_synthesis(*hp, P, d_gmap, d_w, 1, st));
    return CUHPX_OK;
}

int cuhpx_map2alm_iter(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dt, const void* d_map, void* d_alm,
                       const double* d_w, int n_iter, void* d_scratch_map, void* d_scratch_alm, void* ws,
                       size_t ws_bytes, cuhpx_stream_t stream) {
    PlanRef hp;
    int rc = check_call(&hp, nside, lmax, mmax, batch, dt, d_map, MAP, d_alm, ALM, ws, ws_bytes);
    if (rc) return rc;
    if (d_w && ((uintptr_t)d_w & 7)) return CUHPX_EINVAL;
    if (n_iter < 0) return CUHPX_EINVAL;
    if (n_iter > 0) {
        PlanRef h2;
        if ((rc = check_call(&h2, nside, lmax, mmax, batch, dt, d_scratch_map, MAP, d_scratch_alm, ALM, ws, ws_bytes))) return rc;
        if (overlap(d_scratch_map, map_bytes(*hp), d_map, map_bytes(*hp)) ||
            overlap(d_scratch_alm, alm_bytes(*hp), d_alm, alm_bytes(*hp)) ||
            overlap(d_scratch_map, map_bytes(*hp), d_alm, alm_bytes(*hp)) ||
            overlap(d_scratch_alm, alm_bytes(*hp), d_map, map_bytes(*hp)))
            return CUHPX_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const DevPlan P = hp->resolve(ws);
    // a^(0) = A f
    CUDA_OR_FAIL(launch_fft_analysis(*hp, P, d_map, d_w, 1, st));
    CUDA_OR_FAIL(launch_legendre_analysis(*hp, P, d_alm, 0, st));
    const size_t nmap = (size_t)P.batch * (size_t)P.npix, nalm2 = 2 * (size_t)P.batch * (size_t)P.nalm;
    for (int k = 0; k < n_iter; ++k) {
        // r = f - S a
        CUDA_OR_FAIL(launch_legendre_synthesis(*hp, P, d_alm, 0, st));
        CUDA_OR_FAIL(launch_fft_synthesis(*hp, P, d_scratch_map, nullptr, 0, st));
        CUDA_OR_FAIL(launch_residual(dt, d_map, d_scratch_map, nmap, st));
        // a += A r
        CUDA_OR_FAIL(launch_fft_analysis(*hp, P, d_scratch_map, d_w, 1, st));
        CUDA_OR_FAIL(launch_legendre_analysis(*hp, P, d_scratch_alm, 0, st));
        CUDA_OR_FAIL(launch_accumulate(dt, d_scratch_alm, d_alm, nalm2, st));
    }
    return CUHPX_OK;
}

// ---- iso-latitude grids: the same two stages on another ring table
size_t cuhpx_grid_npix(int grid, int nlat, int nlon) {
    const Grid g{grid, nlat, grid == CUHPX_GRID_HEALPIX ? 0 : nlon};
    if (!valid_grid(g)) return 0;
    return grid == CUHPX_GRID_HEALPIX ? (size_t)12 * nlat * nlat : (size_t)nlat * nlon;
}

int cuhpx_grid_ring_info(int grid, int nlat, int nlon, int ring, double* cos_theta, double* weight) {
    const Grid g{grid, nlat, nlon};
    if (grid == CUHPX_GRID_HEALPIX || !valid_grid(g) || ring < 1 || ring > nlat) return CUHPX_EINVAL;
    std::vector<ld> th, w;
    if (grid == CUHPX_GRID_GAUSS_LEGENDRE) gauss_legendre(nlat, th, w);
    else fejer1(nlat, th, w);
    if (cos_theta) *cos_theta = (double)cosl(th[ring - 1]);
    if (weight) *weight = (double)(w[ring - 1] * 2 * PI_LD / (ld)nlon);
    return CUHPX_OK;
}

size_t cuhpx_grid_workspace_bytes(int grid, int nlat, int nlon, int lmax, int mmax, int batch, cuhpx_dtype_t dtype) {
    const Grid g{grid, nlat, grid == CUHPX_GRID_HEALPIX ? 0 : nlon};
    if (!valid_call(g, lmax, mmax, batch, dtype) || !fft_supported(grid_max_ring(g), dtype)) return 0;
    return get_plan(g, lmax, mmax, batch, dtype)->workspace_bytes;
}

int cuhpx_grid_workspace_init(int grid, int nlat, int nlon, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, void* ws,
                              size_t ws_bytes, cuhpx_stream_t stream) {
    return workspace_init_impl(Grid{grid, nlat, grid == CUHPX_GRID_HEALPIX ? 0 : nlon}, lmax, mmax, batch, dtype, ws, ws_bytes, stream);
}

// op: 0 alm2map, 1 map2alm, 2 alm2map_adjoint, 3 map2alm_adjoint
static int grid_op(int op, int grid, int nlat, int nlon, int lmax, int mmax, int batch, cuhpx_dtype_t dt, const void* in, void* out,
                   const double* d_w, void* ws, size_t ws_bytes, cuhpx_stream_t stream) {
    const Grid g{grid, nlat, grid == CUHPX_GRID_HEALPIX ? 0 : nlon};
    const bool in_is_map = op == 1 || op == 2;
    PlanRef hp;
    int rc = check_call(&hp, g, lmax, mmax, batch, dt, in, in_is_map ? MAP : ALM, out, in_is_map ? ALM : MAP, ws, ws_bytes);
    if (rc) return rc;
    if (d_w && ((uintptr_t)d_w & 7)) return CUHPX_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const DevPlan P = hp->resolve(ws);
    switch (op) {
        case 0:
            CUDA_OR_FAIL(launch_legendre_synthesis(*hp, P, in, 0, st));
            CUDA_OR_FAIL(launch_fft_synthesis(*hp, P, out, nullptr, 0, st));
            break;
        case 1:
            CUDA_OR_FAIL(launch_fft_analysis(*hp, P, in, d_w, 1, st));
            CUDA_OR_FAIL(launch_legendre_analysis(*hp, P, out, 0, st));
            break;
        case 2:
            CUDA_OR_FAIL(launch_fft_analysis(*hp, P, in, nullptr, 0, st));
            CUDA_OR_FAIL(launch_legendre_analysis(*hp, P, out, 1, st));
            break;
        default:
            CUDA_OR_FAIL(launch_legendre_synthesis(*hp, P, in, 1, st));
            CUDA_OR_FAIL(launch_fft_synthesis(*hp, P, out, d_w, 1, st));
            break;
    }
    return CUHPX_OK;
}

int cuhpx_grid_alm2map(int grid, int nlat, int nlon, int lmax, int mmax, int batch, cuhpx_dtype_t dt, const void* d_alm, void* d_map,
                       void* ws, size_t ws_bytes, cuhpx_stream_t stream) {
    return grid_op(0, grid, nlat, nlon, lmax, mmax, batch, dt, d_alm, d_map, nullptr, ws, ws_bytes, stream);
}
int cuhpx_grid_map2alm(int grid, int nlat, int nlon, int lmax, int mmax, int batch, cuhpx_dtype_t dt, const void* d_map, void* d_alm,
                       const double* d_w, void* ws, size_t ws_bytes, cuhpx_stream_t stream) {
    return grid_op(1, grid, nlat, nlon, lmax, mmax, batch, dt, d_map, d_alm, d_w, ws, ws_bytes, stream);
}
int cuhpx_grid_alm2map_adjoint(int grid, int nlat, int nlon, int lmax, int mmax, int batch, cuhpx_dtype_t dt, const void* d_gmap,
                               void* d_galm, void* ws, size_t ws_bytes, cuhpx_stream_t stream) {
    return grid_op(2, grid, nlat, nlon, lmax, mmax, batch, dt, d_gmap, d_galm, nullptr, ws, ws_bytes, stream);
}
int cuhpx_grid_map2alm_adjoint(int grid, int nlat, int nlon, int lmax, int mmax, int batch, cuhpx_dtype_t dt, const void* d_galm,
                               void* d_gmap, const double* d_w, void* ws, size_t ws_bytes, cuhpx_stream_t stream) {
    return grid_op(3, grid, nlat, nlon, lmax, mmax, batch, dt, d_galm, d_gmap, d_w, ws, ws_bytes, stream);
}

static int ring_weights_lmax(int nside, int lmax_w) { return lmax_w > 0 ? lmax_w : 3 * nside; }

size_t cuhpx_ring_weights_workspace_bytes(int nside, int lmax_w) {
    const int lw = ring_weights_lmax(nside, lmax_w);
    if (!valid_args(nside, lw, 0, 1, CUHPX_F64) || lw > 3 * nside || !fft_supported(4 * nside, CUHPX_F64)) return 0;
    return ring_weights_scratch_bytes(get_plan(nside, lw, 0, 1, CUHPX_F64)->workspace_bytes, lw);
}

int cuhpx_ring_weights(int nside, int lmax_w, double* d_weights, void* ws, size_t ws_bytes, cuhpx_stream_t stream) {
    const int lw = ring_weights_lmax(nside, lmax_w);
    if (!valid_args(nside, lw, 0, 1, CUHPX_F64) || lw > 3 * nside) return CUHPX_EINVAL;
    if (!d_weights || !ws || ((uintptr_t)d_weights & 7) || ((uintptr_t)ws & 15)) return CUHPX_EINVAL;
    if (!fft_supported(4 * nside, CUHPX_F64)) return CUHPX_EUNSUPPORTED;
    PlanRef hp = get_plan(nside, lw, 0, 1, CUHPX_F64);
    const size_t need = ring_weights_scratch_bytes(hp->workspace_bytes, lw);
    if (ws_bytes < need) return CUHPX_EWORKSPACE;
    if (overlap(d_weights, sizeof(double) * (size_t)hp->d.nrings, ws, need)) return CUHPX_EINVAL;
    const int rc = cuhpx_workspace_init(nside, lw, 0, 1, CUHPX_F64, ws, hp->workspace_bytes, stream);
    if (rc != CUHPX_OK) return rc;
    double resid = 0.0;
    char* vec = (char*)ws + (hp->workspace_bytes + 255) / 256 * 256;
    CUDA_OR_FAIL(ring_weights_solve(*hp, hp->resolve(ws), vec, d_weights, &resid, (cudaStream_t)stream));
    // the constraints hold to rounding when the conjugate gradients have converged (they do for lmax_w <= 3 nside)
    return resid <= 1e-11 ? CUHPX_OK : CUHPX_EUNSUPPORTED;
}

int cuhpx_reorder(int nside, int batch, cuhpx_dtype_t dt, int direction, const void* d_in, void* d_out,
                  cuhpx_stream_t stream) {
    if (nside < 1 || !is_pow2(nside) || nside > (1 << 13) || batch < 1 || batch > MAX_BATCH || (dt != CUHPX_F32 && dt != CUHPX_F64))
        return CUHPX_EINVAL;
    if (direction != CUHPX_NEST2RING && direction != CUHPX_RING2NEST) return CUHPX_EINVAL;
    if (!d_in || !d_out || ((uintptr_t)d_in & 15) || ((uintptr_t)d_out & 15)) return CUHPX_EINVAL;
    const size_t nb = (size_t)batch * 12 * nside * nside * (dt == CUHPX_F64 ? 8 : 4);
    if (overlap(d_in, nb, d_out, nb)) return CUHPX_EINVAL;
    CUDA_OR_FAIL(launch_reorder(nside, batch, dt, direction == CUHPX_NEST2RING, d_in, d_out, (cudaStream_t)stream));
    return CUHPX_OK;
}

int cuhpx_reorder_layout(int nside, int batch, cuhpx_dtype_t dt, int src_layout, int dst_layout, const void* d_in, void* d_out,
                         cuhpx_stream_t stream) {
    if (nside < 1 || !is_pow2(nside) || nside > (1 << 13) || batch < 1 || batch > MAX_BATCH || (dt != CUHPX_F32 && dt != CUHPX_F64))
        return CUHPX_EINVAL;
    if (src_layout < 0 || src_layout > 9 || dst_layout < 0 || dst_layout > 9) return CUHPX_EINVAL;
    if (!d_in || !d_out || ((uintptr_t)d_in & 15) || ((uintptr_t)d_out & 15)) return CUHPX_EINVAL;
    const size_t nb = (size_t)batch * 12 * nside * nside * (dt == CUHPX_F64 ? 8 : 4);
    if (overlap(d_in, nb, d_out, nb)) return CUHPX_EINVAL;
    CUDA_OR_FAIL(launch_layout(nside, batch, dt, src_layout, dst_layout, d_in, d_out, (cudaStream_t)stream));
    return CUHPX_OK;
}

long long cuhpx_layout_index(int nside, int src_layout, int dst_layout, long long ip_src) {
    if (nside < 1 || !is_pow2(nside) || nside > (1 << 13) || ip_src < 0 || ip_src >= 12LL * nside * nside) return -1;
    if (src_layout < 1 || src_layout > 9 || dst_layout < 0 || dst_layout > 9) return -1;
    return layout_index(nside, src_layout, dst_layout, ip_src);
}

int cuhpx_alm_resize(int lmax_in, int mmax_in, int lmax_out, int mmax_out, int batch, cuhpx_dtype_t dt,
                     const void* d_in, void* d_out, cuhpx_stream_t stream) {
    if (lmax_in < 0 || mmax_in < 0 || mmax_in > lmax_in || lmax_out < 0 || mmax_out < 0 || mmax_out > lmax_out) return CUHPX_EINVAL;
    if (batch < 1 || batch > MAX_BATCH || (dt != CUHPX_F32 && dt != CUHPX_F64)) return CUHPX_EINVAL;
    if (!d_in || !d_out || ((uintptr_t)d_in & 15) || ((uintptr_t)d_out & 15)) return CUHPX_EINVAL;
    const size_t cs = dt == CUHPX_F64 ? 16 : 8;
    if (overlap(d_in, batch * cuhpx_alm_count(lmax_in, mmax_in) * cs, d_out, batch * cuhpx_alm_count(lmax_out, mmax_out) * cs))
        return CUHPX_EINVAL;
    CUDA_OR_FAIL(launch_alm_resize(lmax_in, mmax_in, lmax_out, mmax_out, batch, dt, d_in, d_out, (cudaStream_t)stream));
    return CUHPX_OK;
}

long long cuhpx_nest2ring_index(int nside, long long ipnest) {
    if (nside < 1 || !is_pow2(nside) || nside > (1 << 13) || ipnest < 0 || ipnest >= 12LL * nside * nside) return -1;
    return nest_to_ring_index(nside, ipnest);
}

int cuhpx_fma_peak_probe(cuhpx_dtype_t dt, int iters, float* ms, double* fma_count, cuhpx_stream_t stream) {
    if ((dt != CUHPX_F32 && dt != CUHPX_F64) || iters < 1 || !ms || !fma_count) return CUHPX_EINVAL;
    CUDA_OR_FAIL(fma_peak_probe(dt, iters, ms, fma_count, (cudaStream_t)stream));
    return CUHPX_OK;
}

}  // extern "C"

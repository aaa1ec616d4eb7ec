// Host side of libcuhpx.so: argument validation, HEALPix ring geometry, seed / cut-off
// tables, workspace carve-up, the workspace registry and the extern "C" entry points of include/cuhpx.h.
#include <cuda_runtime.h>
#include <math.h>
#include <string.h>

#include <map>
#include <mutex>
#include <vector>

#include "cuhpx_internal.h"

namespace cuhpx {

int legendre_chunk_pairs(cuhpx_dtype_t dt, int batch, int lmax, int npairs);  // legendre.cu

namespace {

typedef long double ld;
const ld PI_LD = 3.14159265358979323846264338327950288419716939937510L;

std::mutex g_mu;
std::map<void*, HostPlan*> g_plans;

bool valid_args(int nside, int lmax, int mmax, int batch, int dtype) {
    if (nside < 1 || nside > (1 << 13) || !is_pow2(nside)) return false;
    if (lmax < 0 || mmax < 0 || mmax > lmax || lmax > 4 * (1 << 13)) return false;
    if (batch < 1 || batch > (1 << 20)) return false;
    if (dtype != CUHPX_F32 && dtype != CUHPX_F64) return false;
    return true;
}

// Gorski et al. ring table, northern hemisphere incl. equator: ring pair j (0-based) <-> ring i = j + 1.
struct PairGeom {
    int N;
    long long start;
    int shifted;
    ld y;    // 1 - cos(theta), exact rational rounded once
    ld sth;  // sin(theta)
};

PairGeom pair_geom(int nside, int j) {
    PairGeom g;
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

struct Layout {
    size_t off_y, off_lshi, off_lslo, off_ringN, off_start, off_shifted, off_mcut, off_prefhi, off_preflo, off_jmin;
    size_t off_fft, fft_bytes, off_alpha, off_scale, off_spectra, off_partial, total;
};

Layout make_layout(HostPlan& hp) {
    DevPlan& d = hp.d;
    Layout L;
    size_t o = 256;  // header
    auto take = [&](size_t bytes) {
        size_t r = o;
        o = align_up(o + bytes);
        return r;
    };
    L.off_y = take(sizeof(double) * d.npairs);
    L.off_lshi = take(sizeof(double) * d.npairs);
    L.off_lslo = take(sizeof(double) * d.npairs);
    L.off_ringN = take(sizeof(int) * d.npairs);
    L.off_start = take(sizeof(long long) * d.npairs);
    L.off_shifted = take(sizeof(int) * d.npairs);
    L.off_mcut = take(sizeof(int) * d.npairs);
    L.off_prefhi = take(sizeof(double) * (d.mmax + 1));
    L.off_preflo = take(sizeof(double) * (d.mmax + 1));
    L.off_jmin = take(sizeof(int) * (d.mmax + 1));
    L.off_fft = o;
    cudaError_t err = cudaSuccess;
    L.fft_bytes = plan_fft_tables(hp, nullptr, false, nullptr, &err);
    o = align_up(o + L.fft_bytes);
    L.off_alpha = take(sizeof(double) * (size_t)d.nalm);
    L.off_scale = take(sizeof(double) * (size_t)d.nalm);
    const size_t csize = hp.dtype == CUHPX_F64 ? 16 : 8;
    L.off_spectra = take(csize * (size_t)d.batch * d.nrings * d.mstride);
    L.off_partial = o;
    if (d.nchunk_max > 1) take(csize * (size_t)d.nchunk_max * d.batch * d.nalm);
    L.total = o;
    return L;
}

void fill_basic(HostPlan& hp, int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dt) {
    DevPlan& d = hp.d;
    memset(&d, 0, sizeof(d));
    hp.dtype = dt;
    d.nside = nside;
    d.lmax = lmax;
    d.mmax = mmax;
    d.batch = batch;
    d.nrings = 4 * nside - 1;
    d.npairs = 2 * nside;
    d.mstride = (int)cuhpx_spectra_stride(mmax);
    d.npix = 12LL * nside * nside;
    d.nalm = (long long)cuhpx_alm_count(lmax, mmax);
    d.chunk_pairs = legendre_chunk_pairs(dt, batch, lmax, d.npairs);
    d.nchunk_max = (d.npairs + d.chunk_pairs - 1) / d.chunk_pairs;
    hp.h_ringN.resize(d.npairs);
    hp.h_start.resize(d.npairs);
    hp.h_shifted.resize(d.npairs);
    for (int j = 0; j < d.npairs; ++j) {
        PairGeom g = pair_geom(nside, j);
        hp.h_ringN[j] = g.N;
        hp.h_start[j] = g.start;
        hp.h_shifted[j] = g.shifted;
    }
}

HostPlan* find_plan(void* ws) {
    std::lock_guard<std::mutex> lk(g_mu);
    auto it = g_plans.find(ws);
    return it == g_plans.end() ? nullptr : it->second;
}

int check_call(HostPlan** out, int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dt, const void* a,
               const void* b, void* ws, size_t ws_bytes) {
    if (!valid_args(nside, lmax, mmax, batch, dt)) return CUHPX_EINVAL;
    if (!a || !b || !ws) return CUHPX_EINVAL;
    if (((uintptr_t)a & 15) || ((uintptr_t)b & 15) || ((uintptr_t)ws & 15)) return CUHPX_EINVAL;
    if (a == b) return CUHPX_EINVAL;
    HostPlan* hp = find_plan(ws);
    if (!hp) return CUHPX_EWORKSPACE;
    const DevPlan& d = hp->d;
    if (d.nside != nside || d.lmax != lmax || d.mmax != mmax || d.batch != batch || hp->dtype != dt)
        return CUHPX_EWORKSPACE;
    if (ws_bytes < hp->workspace_bytes) return CUHPX_EWORKSPACE;
    *out = hp;
    return CUHPX_OK;
}

}  // namespace
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
        case CUHPX_EINVAL: return "CUHPX_EINVAL: bad nside/lmax/mmax/batch/dtype or null/misaligned/aliased pointer";
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
    if (!valid_args(nside, lmax, mmax, batch, dtype) || !fft_supported(nside, dtype)) return 0;
    HostPlan hp;
    fill_basic(hp, nside, lmax, mmax, batch, dtype);
    return make_layout(hp).total;
}

int cuhpx_workspace_init(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, void* ws, size_t ws_bytes,
                         cuhpx_stream_t stream) {
    if (!valid_args(nside, lmax, mmax, batch, dtype)) return CUHPX_EINVAL;
    if (!ws || ((uintptr_t)ws & 15)) return CUHPX_EINVAL;
    if (!fft_supported(nside, dtype)) return CUHPX_EUNSUPPORTED;
    HostPlan* hp = new HostPlan;
    fill_basic(*hp, nside, lmax, mmax, batch, dtype);
    Layout L = make_layout(*hp);
    hp->workspace_bytes = L.total;
    if (ws_bytes < L.total) {
        delete hp;
        return CUHPX_EWORKSPACE;
    }
    DevPlan& d = hp->d;
    char* base = (char*)ws;
    cudaStream_t st = (cudaStream_t)stream;

    // ---- per-pair and per-m tables (long double on the host)
    std::vector<double> y(d.npairs), lshi(d.npairs), lslo(d.npairs), prefhi(mmax + 1), preflo(mmax + 1);
    std::vector<ld> lg2sin(d.npairs), pref(mmax + 1);
    for (int j = 0; j < d.npairs; ++j) {
        PairGeom g = pair_geom(nside, j);
        y[j] = (double)g.y;
        lg2sin[j] = log2l(g.sth);
        split_hi_lo(lg2sin[j], lshi[j], lslo[j]);
    }
    // log2 |lambda_mm| = -0.5 log2(4 pi) + 0.5 sum_{k<=m} log2(1 + 1/(2k)) + m log2 sin(theta)   (Eq. 15)
    ld acc = -0.5L * log2l(4.0L * PI_LD);
    for (int m = 0; m <= mmax; ++m) {
        if (m > 0) acc += 0.5L * log1pl(1.0L / (2.0L * m)) / logl(2.0L);
        pref[m] = acc;
        split_hi_lo(acc, prefhi[m], preflo[m]);
    }
    // ---- jmin[m]: first ring pair that matters at order m (two-pointer: the active set shrinks with m)
    hp->h_jmin.assign(mmax + 1, 0);
    int j = 0;
    for (int m = 0; m <= mmax; ++m) {
        while (j < d.npairs - 1 && !pair_active(lmax, m, pref[m], lg2sin[j], y[j])) ++j;
        hp->h_jmin[m] = j;
    }
    // ---- mcut[j]: last order at which pair j is processed
    hp->h_mcut.assign(d.npairs, 0);
    {
        int m = mmax;
        for (int jj = d.npairs - 1; jj >= 0; --jj) {
            while (m > 0 && hp->h_jmin[m] > jj) --m;
            hp->h_mcut[jj] = m;
        }
        // make it monotone non-decreasing in j as the sweep implies
    }

    cudaError_t e = cudaSuccess;
    auto up = [&](size_t off, const void* src, size_t bytes) {
        if (e == cudaSuccess) e = cudaMemcpyAsync(base + off, src, bytes, cudaMemcpyHostToDevice, st);
    };
    up(L.off_y, y.data(), sizeof(double) * d.npairs);
    up(L.off_lshi, lshi.data(), sizeof(double) * d.npairs);
    up(L.off_lslo, lslo.data(), sizeof(double) * d.npairs);
    up(L.off_ringN, hp->h_ringN.data(), sizeof(int) * d.npairs);
    up(L.off_start, hp->h_start.data(), sizeof(long long) * d.npairs);
    up(L.off_shifted, hp->h_shifted.data(), sizeof(int) * d.npairs);
    up(L.off_mcut, hp->h_mcut.data(), sizeof(int) * d.npairs);
    up(L.off_prefhi, prefhi.data(), sizeof(double) * (mmax + 1));
    up(L.off_preflo, preflo.data(), sizeof(double) * (mmax + 1));
    up(L.off_jmin, hp->h_jmin.data(), sizeof(int) * (mmax + 1));
    // pageable sources: make sure the copies are done before the vectors die
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);

    d.y = (const double*)(base + L.off_y);
    d.ls_hi = (const double*)(base + L.off_lshi);
    d.ls_lo = (const double*)(base + L.off_lslo);
    d.ringN = (const int*)(base + L.off_ringN);
    d.start = (const long long*)(base + L.off_start);
    d.shifted = (const int*)(base + L.off_shifted);
    d.mcut = (const int*)(base + L.off_mcut);
    d.pref_hi = (const double*)(base + L.off_prefhi);
    d.pref_lo = (const double*)(base + L.off_preflo);
    d.jmin = (const int*)(base + L.off_jmin);
    d.coef_alpha = (const double*)(base + L.off_alpha);
    d.coef_scale = (const double*)(base + L.off_scale);
    if (e == cudaSuccess)
        e = launch_legendre_coeff(lmax, mmax, (double*)(base + L.off_alpha), (double*)(base + L.off_scale), st);
    d.spectra = base + L.off_spectra;
    d.partial = d.nchunk_max > 1 ? base + L.off_partial : nullptr;

    if (e == cudaSuccess) {
        cudaError_t e2 = cudaSuccess;
        plan_fft_tables(*hp, base + L.off_fft, true, st, &e2);
        e = e2;
    }
    if (e != cudaSuccess) {
        delete hp;
        return CUHPX_ECUDA;
    }
    {
        std::lock_guard<std::mutex> lk(g_mu);
        auto it = g_plans.find(ws);
        if (it != g_plans.end()) {
            delete it->second;
            g_plans.erase(it);
        }
        g_plans[ws] = hp;
    }
    return CUHPX_OK;
}

int cuhpx_workspace_release(void* ws) {
    std::lock_guard<std::mutex> lk(g_mu);
    auto it = g_plans.find(ws);
    if (it == g_plans.end()) return CUHPX_EWORKSPACE;
    delete it->second;
    g_plans.erase(it);
    return CUHPX_OK;
}

void* cuhpx_workspace_spectra(void* ws) {
    HostPlan* hp = find_plan(ws);
    return hp ? hp->d.spectra : nullptr;
}

int cuhpx_workspace_mcut(void* ws, int* h_mcut) {
    HostPlan* hp = find_plan(ws);
    if (!hp || !h_mcut) return CUHPX_EWORKSPACE;
    const DevPlan& d = hp->d;
    for (int r = 0; r < d.nrings; ++r) {
        const int j = r < d.nrings - 1 - r ? r : d.nrings - 1 - r;
        h_mcut[r] = hp->h_mcut[j];
    }
    return CUHPX_OK;
}

int cuhpx_workspace_stats(void* ws, double* out, int count) {
    HostPlan* hp = find_plan(ws);
    if (!hp || !out || count < 1) return CUHPX_EWORKSPACE;
    const DevPlan& d = hp->d;
    double st[8] = {0};
    int fl = 0;
    double tb = 0;
    fft_stage_stats(*hp, &fl, &tb);
    st[0] = fl;
    st[1] = d.nchunk_max > 1 ? 2 : 1;
    st[2] = 1;
    for (int m = 0; m <= d.mmax; ++m) st[3] += (double)(d.lmax - m + 1) * (double)(d.npairs - hp->h_jmin[m]);
    st[4] = (double)d.nalm * (double)d.npairs;
    for (int r = 0; r < d.nrings; ++r) st[5] += hp->h_mcut[r < d.nrings - 1 - r ? r : d.nrings - 1 - r] + 1;
    st[6] = tb;
    st[7] = (double)hp->workspace_bytes;
    for (int i = 0; i < count && i < 8; ++i) out[i] = st[i];
    return CUHPX_OK;
}

#define CUDA_OR_FAIL(expr)                         \
    do {                                           \
        if ((expr) != cudaSuccess) return CUHPX_ECUDA; \
    } while (0)

int cuhpx_analysis_fft_stage(const void* d_map, const double* d_w, int use_w, void* ws, cuhpx_stream_t stream) {
    HostPlan* hp = find_plan(ws);
    if (!hp) return CUHPX_EWORKSPACE;
    if (!d_map) return CUHPX_EINVAL;
    CUDA_OR_FAIL(launch_fft_analysis(*hp, d_map, d_w, use_w, (cudaStream_t)stream));
    return CUHPX_OK;
}

int cuhpx_analysis_legendre_stage(void* d_alm, int adjoint, void* ws, cuhpx_stream_t stream) {
    HostPlan* hp = find_plan(ws);
    if (!hp) return CUHPX_EWORKSPACE;
    if (!d_alm) return CUHPX_EINVAL;
    CUDA_OR_FAIL(launch_legendre_analysis(*hp, d_alm, adjoint, (cudaStream_t)stream));
    return CUHPX_OK;
}

int cuhpx_synthesis_legendre_stage(const void* d_alm, int adjoint, void* ws, cuhpx_stream_t stream) {
    HostPlan* hp = find_plan(ws);
    if (!hp) return CUHPX_EWORKSPACE;
    if (!d_alm) return CUHPX_EINVAL;
    CUDA_OR_FAIL(launch_legendre_synthesis(*hp, d_alm, adjoint, (cudaStream_t)stream));
    return CUHPX_OK;
}

int cuhpx_synthesis_fft_stage(void* d_map, const double* d_w, int use_w, void* ws, cuhpx_stream_t stream) {
    HostPlan* hp = find_plan(ws);
    if (!hp) return CUHPX_EWORKSPACE;
    if (!d_map) return CUHPX_EINVAL;
    CUDA_OR_FAIL(launch_fft_synthesis(*hp, d_map, d_w, use_w, (cudaStream_t)stream));
    return CUHPX_OK;
}

int cuhpx_map2alm(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dt, const void* d_map, void* d_alm,
                  const double* d_w, void* ws, size_t ws_bytes, cuhpx_stream_t stream) {
    HostPlan* hp = nullptr;
    int rc = check_call(&hp, nside, lmax, mmax, batch, dt, d_map, d_alm, ws, ws_bytes);
    if (rc) return rc;
    if (d_w && ((uintptr_t)d_w & 7)) return CUHPX_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_OR_FAIL(launch_fft_analysis(*hp, d_map, d_w, 1, st));
    CUDA_OR_FAIL(launch_legendre_analysis(*hp, d_alm, 0, st));
    return CUHPX_OK;
}

int cuhpx_alm2map_adjoint(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dt, const void* d_gmap,
                          void* d_galm, void* ws, size_t ws_bytes, cuhpx_stream_t stream) {
    HostPlan* hp = nullptr;
    int rc = check_call(&hp, nside, lmax, mmax, batch, dt, d_gmap, d_galm, ws, ws_bytes);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_OR_FAIL(launch_fft_analysis(*hp, d_gmap, nullptr, 0, st));
    CUDA_OR_FAIL(launch_legendre_analysis(*hp, d_galm, 1, st));
    return CUHPX_OK;
}

int cuhpx_alm2map(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dt, const void* d_alm, void* d_map,
                  void* ws, size_t ws_bytes, cuhpx_stream_t stream) {
    HostPlan* hp = nullptr;
    int rc = check_call(&hp, nside, lmax, mmax, batch, dt, d_alm, d_map, ws, ws_bytes);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_OR_FAIL(launch_legendre_synthesis(*hp, d_alm, 0, st));
    CUDA_OR_FAIL(launch_fft_synthesis(*hp, d_map, nullptr, 0, st));
    return CUHPX_OK;
}

int cuhpx_map2alm_adjoint(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dt, const void* d_galm,
                          void* d_gmap, const double* d_w, void* ws, size_t ws_bytes, cuhpx_stream_t stream) {
    HostPlan* hp = nullptr;
    int rc = check_call(&hp, nside, lmax, mmax, batch, dt, d_galm, d_gmap, ws, ws_bytes);
    if (rc) return rc;
    if (d_w && ((uintptr_t)d_w & 7)) return CUHPX_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_OR_FAIL(launch_legendre_synthesis(*hp, d_galm, 1, st));
    CUDA_OR_FAIL(launch_fft_synthesis(*hp, d_gmap, d_w, 1, st));
    return CUHPX_OK;
}

int cuhpx_map2alm_iter(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dt, const void* d_map, void* d_alm,
                       const double* d_w, int n_iter, void* d_scratch_map, void* d_scratch_alm, void* ws,
                       size_t ws_bytes, cuhpx_stream_t stream) {
    HostPlan* hp = nullptr;
    int rc = check_call(&hp, nside, lmax, mmax, batch, dt, d_map, d_alm, ws, ws_bytes);
    if (rc) return rc;
    if (d_w && ((uintptr_t)d_w & 7)) return CUHPX_EINVAL;
    if (n_iter < 0) return CUHPX_EINVAL;
    if (n_iter > 0 && (!d_scratch_map || !d_scratch_alm || ((uintptr_t)d_scratch_map & 15) || ((uintptr_t)d_scratch_alm & 15) ||
                       d_scratch_map == d_map || d_scratch_alm == d_alm))
        return CUHPX_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    // a^(0) = A f
    CUDA_OR_FAIL(launch_fft_analysis(*hp, d_map, d_w, 1, st));
    CUDA_OR_FAIL(launch_legendre_analysis(*hp, d_alm, 0, st));
    const size_t nmap = (size_t)hp->d.batch * (size_t)hp->d.npix, nalm2 = 2 * (size_t)hp->d.batch * (size_t)hp->d.nalm;
    for (int k = 0; k < n_iter; ++k) {
        // r = f - S a
        CUDA_OR_FAIL(launch_legendre_synthesis(*hp, d_alm, 0, st));
        CUDA_OR_FAIL(launch_fft_synthesis(*hp, d_scratch_map, nullptr, 0, st));
        CUDA_OR_FAIL(launch_residual(dt, d_map, d_scratch_map, nmap, st));
        // a += A r
        CUDA_OR_FAIL(launch_fft_analysis(*hp, d_scratch_map, d_w, 1, st));
        CUDA_OR_FAIL(launch_legendre_analysis(*hp, d_scratch_alm, 0, st));
        CUDA_OR_FAIL(launch_accumulate(dt, d_scratch_alm, d_alm, nalm2, st));
    }
    return CUHPX_OK;
}

int cuhpx_reorder(int nside, int batch, cuhpx_dtype_t dt, int direction, const void* d_in, void* d_out,
                  cuhpx_stream_t stream) {
    if (nside < 1 || !is_pow2(nside) || nside > (1 << 13) || batch < 1 || (dt != CUHPX_F32 && dt != CUHPX_F64)) return CUHPX_EINVAL;
    if (direction != CUHPX_NEST2RING && direction != CUHPX_RING2NEST) return CUHPX_EINVAL;
    if (!d_in || !d_out || d_in == d_out || ((uintptr_t)d_in & 15) || ((uintptr_t)d_out & 15)) return CUHPX_EINVAL;
    CUDA_OR_FAIL(launch_reorder(nside, batch, dt, direction == CUHPX_NEST2RING, d_in, d_out, (cudaStream_t)stream));
    return CUHPX_OK;
}

int cuhpx_alm_resize(int lmax_in, int mmax_in, int lmax_out, int mmax_out, int batch, cuhpx_dtype_t dt,
                     const void* d_in, void* d_out, cuhpx_stream_t stream) {
    if (lmax_in < 0 || mmax_in < 0 || mmax_in > lmax_in || lmax_out < 0 || mmax_out < 0 || mmax_out > lmax_out) return CUHPX_EINVAL;
    if (batch < 1 || (dt != CUHPX_F32 && dt != CUHPX_F64)) return CUHPX_EINVAL;
    if (!d_in || !d_out || d_in == d_out || ((uintptr_t)d_in & 15) || ((uintptr_t)d_out & 15)) return CUHPX_EINVAL;
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

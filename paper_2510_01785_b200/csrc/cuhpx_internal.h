// Internal declarations shared by the host planner and the CUDA kernels of libcuhpx.so.
// (Product code: shares nothing with oracle/.)
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include <memory>
#include <vector>

#include "../../include/cuhpx.h"

namespace cuhpx {

// ------------------------------------------------------------------ workspace header (first 256 bytes of a workspace)
// Written by cuhpx_workspace_init after every table is in place; every kernel of a transform call checks
// (magic, key) before it touches a table and returns without side effects other than `bad = 1` if they do not
// match.  The host keeps nothing per workspace: tables are addressed as workspace base + offset, and the offsets
// are a pure function of (nside, lmax, mmax, batch, dtype, geometry).
constexpr unsigned long long WS_MAGIC = 0x6375485058763032ULL;  // "cuHPXv02"
struct WsHeader {
    unsigned long long magic;
    unsigned long long key;  // plan_key(nside, lmax, mmax, batch, dtype, geometry)
    int nside, lmax, mmax, batch, dtype, geometry;
    unsigned long long bytes;
    int bad;  // set by a kernel that found a foreign header
    int pad;
};
static_assert(sizeof(WsHeader) <= 256, "header slot");

inline unsigned long long plan_key(int nside, int lmax, int mmax, int batch, int dtype, int geometry) {
    unsigned long long h = 0x9E3779B97F4A7C15ULL;
    const int v[6] = {nside, lmax, mmax, batch, dtype, geometry};
    for (int i = 0; i < 6; ++i) {
        h ^= (unsigned long long)(unsigned)v[i] + 0x9E3779B97F4A7C15ULL + (h << 6) + (h >> 2);
        h *= 0xBF58476D1CE4E5B9ULL;
    }
    return h | 1ULL;
}

// ------------------------------------------------------------------ device-visible plan (POD, passed by value)
// Ring pairs j = 0 .. npairs-1: north ring index j (0-based ring number = j), its mirror is ring nrings-1-j; when
// nrings is odd the middle ring (j = npairs-1) is its own mirror and is treated as a pair with an empty south
// member.  SURVEY 8(a) a0.  HEALPix: npairs = 2 nside, nrings = 4 nside - 1.
struct DevPlan {
    int nside, lmax, mmax, batch;
    int nrings, npairs;
    int mstride;         // complex values per spectra row
    long long npix, nalm;
    const WsHeader* hdr;     // workspace header (device) and the key this call expects to find there
    unsigned long long key;
    // per ring pair [npairs]
    const double* y;         // 1 - cos(theta_j)  (formed without cancellation; R3)
    const double* ls_hi;     // log2(sin theta_j), split hi + lo
    const double* ls_lo;
    const int* ringN;        // N_j pixels in the ring
    const long long* start;  // RING index of first pixel of the NORTH ring
    const int* shifted;      // 1: phi0 = pi/N, 0: phi0 = 0
    const int* mcut;         // largest m for which this ring pair is processed
    // per m [mmax+1]
    const double* pref_hi;   // log2 |lambda_mm| prefactor, split hi + lo
    const double* pref_lo;
    const int* jmin;         // first ring pair processed for this m
    const double* defw;      // [nrings] quadrature weight per pixel used when the caller passes none; null: 4 pi / npix
    // per (l, m) [nalm], packed like alm: rescaled recurrence coefficients (legendre.cu)
    const double* coef_alpha;
    const double* coef_scale;
    // scratch
    void* spectra;           // [batch][nrings][mstride] complex<T>
    void* partial;           // [nchunk_max][batch][nalm] complex<T> (analysis partial sums), or null
    // tensor-core Legendre kernels (fp32, batch >= 8; legendre_tc.cu): operand images built per call
    const long long* tc_prefix;  // [mmax + 2] stages of 32 degrees before order m
    void* tc_images;             // [channel group][stage] images (alpha + B-operand tiles), or null
    int tc_nb;                   // channels per group (0: tensor-core path not planned)
    int nchunk_max;          // ring-pair chunks per m in the Legendre analysis grid
    int chunk_pairs;         // ring pairs per chunk
    // late-start tables of the fp64 Legendre kernels ([0] analysis, [1] synthesis; legendre.cu "late start"): per order
    // and ring chunk the first 64-degree tile in which a ring pair of the chunk becomes significant, and the recurrence
    // state of every ring pair at the start of that tile.  st_chunk = 0: not planned.
    const double* st_cur[2];   // [mmax + 1][npairs]
    const double* st_prev[2];  // [mmax + 1][npairs]
    const int* st_sc[2];       // [mmax + 1][npairs] exponent window of the stored state
    const int* st_l0[2];       // [mmax + 1][st_nchunk] l - m of the first tile to run
    int st_chunk[2];           // ring pairs per chunk the tables were built for
    int st_nchunk[2];
};

// true if the workspace behind P was initialised for the parameters of this call (one 16-byte load per CTA)
__device__ __forceinline__ bool ws_ok(const DevPlan& P) {
#ifdef __CUDA_ARCH__
    const ulonglong2 h = __ldg(reinterpret_cast<const ulonglong2*>(P.hdr));
    if (h.x == WS_MAGIC && h.y == P.key) return true;
    if (threadIdx.x == 0) const_cast<WsHeader*>(P.hdr)->bad = 1;
    return false;
#else
    return true;
#endif
}

// ------------------------------------------------------------------ host plan: a pure function of the call parameters
struct FftHost;  // FFT-stage part (ring_fft.cu)
void free_fft_host(FftHost*);

struct HostPlan {
    DevPlan d;  // pointer members hold OFFSETS from the workspace base until resolve() rebases them
    cuhpx_dtype_t dtype;
    int geometry;
    int max_ring;  // pixels of the longest ring
    size_t workspace_bytes;
    size_t off_defw = 0;
    // table offsets inside the workspace
    size_t off_y, off_lshi, off_lslo, off_ringN, off_start, off_shifted, off_mcut, off_prefhi, off_preflo, off_jmin;
    size_t off_fft, fft_bytes, off_alpha, off_scale, off_spectra, off_partial, off_tcprefix, off_tcimages;
    size_t off_st[2][4] = {{0, 0, 0, 0}, {0, 0, 0, 0}};  // late-start tables: cur, prev, sc, l0
    std::vector<long long> h_tcprefix;
    std::vector<int> h_ringN, h_mcut, h_jmin, h_shifted;
    std::vector<long long> h_start;
    std::vector<double> h_y, h_lshi, h_lslo, h_prefhi, h_preflo, h_weight;  // h_weight: built-in quadrature weights per ring
    FftHost* fft = nullptr;  // owned
    ~HostPlan() { free_fft_host(fft); }
    HostPlan() = default;
    HostPlan(const HostPlan&) = delete;
    HostPlan& operator=(const HostPlan&) = delete;
    DevPlan resolve(void* ws) const;  // device plan for the workspace at `ws`
};
typedef std::shared_ptr<const HostPlan> PlanRef;

inline int ilog2_ceil(long long v) {
    int k = 0;
    while ((1LL << k) < v) ++k;
    return k;
}
inline bool is_pow2(long long v) { return v > 0 && (v & (v - 1)) == 0; }

// ------------------------------------------------------------------ launchers (each returns a cudaError_t)
// tensor-core Legendre path: channels per group for this (dtype, batch) or 0, and bytes of one stage image
int legendre_tc_group(cuhpx_dtype_t dt, int batch);
size_t legendre_tc_image_bytes(int nb);
cudaError_t launch_legendre_coeff(int lmax, int mmax, double* alpha, double* scale, cudaStream_t st);
cudaError_t launch_legendre_analysis(const HostPlan& hp, const DevPlan& P, void* d_alm, int adjoint, cudaStream_t st);
cudaError_t launch_legendre_synthesis(const HostPlan& hp, const DevPlan& P, const void* d_alm, int adjoint, cudaStream_t st);
cudaError_t launch_fft_analysis(const HostPlan& hp, const DevPlan& P, const void* d_map, const double* d_w, int use_w,
                                cudaStream_t st);
cudaError_t launch_fft_synthesis(const HostPlan& hp, const DevPlan& P, void* d_map, const double* d_w, int use_w,
                                 cudaStream_t st);

// FFT-stage planning (host only): classify the rings, lay the tables out; returns the bytes they take
size_t fft_plan_host(HostPlan& hp);
// build the FFT tables inside the workspace (base = workspace + hp.off_fft)
cudaError_t fft_build_tables(const HostPlan& hp, char* base, cudaStream_t st);
// largest supported ring for this dtype (register / shared-memory bound); used by argument validation
bool fft_supported(int max_ring_pixels, cuhpx_dtype_t dt);

// launches per FFT-stage call and bytes of constant tables it reads
void fft_stage_stats(const HostPlan& hp, int* launches, double* table_bytes);

// elementwise steps of the iterative refinement (Eq. 4): r[i] = f[i] - r[i];  a[i] += d[i]
cudaError_t launch_residual(cuhpx_dtype_t dt, const void* f, void* r, size_t n, cudaStream_t st);
cudaError_t launch_accumulate(cuhpx_dtype_t dt, const void* d, void* a, size_t n, cudaStream_t st);

// layout reordering (reorder.cu)
cudaError_t launch_reorder(int nside, int batch, cuhpx_dtype_t dt, int to_ring, const void* in, void* out, cudaStream_t st);
long long nest_to_ring_index(int nside, long long ipnest);
// generic layout conversion (0 RING, 1 NESTED, 2..9 flat variants); layout_index: src must not be RING
cudaError_t launch_layout(int nside, int batch, cuhpx_dtype_t dt, int src, int dst, const void* in, void* out, cudaStream_t st);
long long layout_index(int nside, int src_layout, int dst_layout, long long ip_src);
cudaError_t launch_alm_resize(int lmax_in, int mmax_in, int lmax_out, int mmax_out, int batch, cuhpx_dtype_t dt,
                              const void* in, void* out, cudaStream_t st);

// ring quadrature weights (ring_weights.cu): scratch layout [transform workspace][CG vectors]; the solve synchronises
size_t ring_weights_scratch_bytes(size_t transform_ws_bytes, int lmax_w);
cudaError_t ring_weights_solve(const HostPlan& hp, const DevPlan& P, char* vec_base, double* d_w, double* h_resid, cudaStream_t st);

cudaError_t fma_peak_probe(cuhpx_dtype_t dt, int iters, float* ms, double* count, cudaStream_t st);

}  // namespace cuhpx

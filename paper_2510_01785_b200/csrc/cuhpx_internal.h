// Internal declarations shared by the host planner and the CUDA kernels of libcuhpx.so.
// (Product code: shares nothing with oracle/.)
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include <vector>

#include "../../include/cuhpx.h"

namespace cuhpx {

// ------------------------------------------------------------------ device-visible plan (POD, passed by value)
// Ring pairs j = 0 .. npairs-1 (npairs = 2 nside): north ring index j (0-based ring number = j), its mirror
// is ring nrings-1-j; the equator (j = npairs-1) is its own mirror and is treated as a pair with an empty
// south member.  SURVEY 8(a) a0.
struct DevPlan {
    int nside, lmax, mmax, batch;
    int nrings, npairs;
    int mstride;         // complex values per spectra row
    long long npix, nalm;
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
    // per (l, m) [nalm], packed like alm: rescaled recurrence coefficients (legendre.cu)
    const double* coef_alpha;
    const double* coef_scale;
    // scratch
    void* spectra;           // [batch][nrings][mstride] complex<T>
    void* partial;           // [nchunk_max][batch][nalm] complex<T> (analysis partial sums), or null
    int nchunk_max;          // ring-pair chunks per m in the Legendre analysis grid
    int chunk_pairs;         // ring pairs per chunk
};

// ------------------------------------------------------------------ host plan
struct FftDev;  // FFT-stage device tables, defined in ring_fft.cu
void free_fft_dev(FftDev*);

struct HostPlan {
    DevPlan d;
    cuhpx_dtype_t dtype;
    size_t workspace_bytes;
    std::vector<int> h_ringN, h_mcut, h_jmin, h_shifted;
    std::vector<long long> h_start;
    // ring lists for the FFT stage, by method (0-based ring numbers over all nrings rings)
    std::vector<int> rings_direct, rings_pow2, rings_blue;
    int* d_rings_direct = nullptr;
    int* d_rings_pow2 = nullptr;
    int* d_rings_blue = nullptr;
    FftDev* fft = nullptr;  // owned
    ~HostPlan() { free_fft_dev(fft); }
    HostPlan() = default;
    HostPlan(const HostPlan&) = delete;
    HostPlan& operator=(const HostPlan&) = delete;
};

inline int ilog2_ceil(long long v) {
    int k = 0;
    while ((1LL << k) < v) ++k;
    return k;
}
inline bool is_pow2(long long v) { return v > 0 && (v & (v - 1)) == 0; }

// ------------------------------------------------------------------ launchers (each returns a cudaError_t)
cudaError_t launch_legendre_coeff(int lmax, int mmax, double* alpha, double* scale, cudaStream_t st);
cudaError_t launch_legendre_analysis(const HostPlan& hp, void* d_alm, int adjoint, cudaStream_t st);
cudaError_t launch_legendre_synthesis(const HostPlan& hp, const void* d_alm, int adjoint, cudaStream_t st);
cudaError_t launch_fft_analysis(const HostPlan& hp, const void* d_map, const double* d_w, int use_w, cudaStream_t st);
cudaError_t launch_fft_synthesis(const HostPlan& hp, void* d_map, const double* d_w, int use_w, cudaStream_t st);

// FFT-stage planning: classify rings, size and build tables.  `base` is the device address where the tables may
// be placed; returns the number of bytes used (when base == nullptr only sizes are computed).
size_t plan_fft_tables(HostPlan& hp, char* base, bool build, cudaStream_t st, cudaError_t* err);
// largest supported ring for this dtype (shared-memory bound); used by argument validation
bool fft_supported(int nside, cuhpx_dtype_t dt);

// launches per FFT-stage call and bytes of constant tables it reads
void fft_stage_stats(const HostPlan& hp, int* launches, double* table_bytes);

// elementwise steps of the iterative refinement (Eq. 4): r[i] = f[i] - r[i];  a[i] += d[i]
cudaError_t launch_residual(cuhpx_dtype_t dt, const void* f, void* r, size_t n, cudaStream_t st);
cudaError_t launch_accumulate(cuhpx_dtype_t dt, const void* d, void* a, size_t n, cudaStream_t st);

// layout reordering (reorder.cu)
cudaError_t launch_reorder(int nside, int batch, cuhpx_dtype_t dt, int to_ring, const void* in, void* out, cudaStream_t st);
long long nest_to_ring_index(int nside, long long ipnest);
cudaError_t launch_alm_resize(int lmax_in, int mmax_in, int lmax_out, int mmax_out, int batch, cuhpx_dtype_t dt,
                              const void* in, void* out, cudaStream_t st);

cudaError_t fma_peak_probe(cuhpx_dtype_t dt, int iters, float* ms, double* count, cudaStream_t st);

}  // namespace cuhpx

// FFT stage of the HEALPix SHT: per-ring real DFT in longitude fused with the
// phi0 phase twist and the m-aliasing rule (m mod N_i) of Eq. 24 / Eq. 26.
//   analysis : F_m(i) = w_i exp(-i m phi0_i) X~_i[m mod N_i],  X_i[k] = sum_x p_x exp(-2 pi i k x / N_i)   (Eq. 13)
//   synthesis: p_x = Re G_0 + 2 sum_{m>=1} Re(G_m exp(+i m (phi0_i + 2 pi x / N_i)))                       (Eq. 24)
// Three kernel families, chosen per ring length:
//   direct   : O(N m_cut) sums for short rings (several cheap rings, no FFT set-up cost)
//   pow2     : shared-memory radix-8/4/2 FFT for N = 2^k (all belt rings and cap rings with i a power of two)
//   bluestein: chirp-z (Eq. 17-23) for the other cap rings, per-ring minimal chirp length, in one SM
#include <cuda_runtime.h>
#include <math.h>

#include "cuhpx_internal.h"

namespace cuhpx {

template <typename T> struct V2;
template <> struct V2<float> { using type = float2; };
template <> struct V2<double> { using type = double2; };

constexpr int DIRECT_MAX_N = 1024;
constexpr int FFT_THREADS = 256;

// exp(sign * i * pi * num / den) from exact integers (num already reduced mod 2 den)
__device__ __forceinline__ void cispi_ratio(long long num, long long den, double sign, double& c, double& s) {
    sincospi((double)num / (double)den, &s, &c);
    s *= sign;
}
__device__ __forceinline__ void cispi_ratio(long long num, long long den, float sign, float& c, float& s) {
    sincospif((float)((double)num / (double)den), &s, &c);
    s *= sign;
}

struct RingRef {
    int N, mcut, shifted;
    long long start;
    double weight;
};

__device__ __forceinline__ RingRef ring_ref(const DevPlan& P, int r, const double* w, int use_w) {
    RingRef R;
    const int j = min(r, P.nrings - 1 - r);
    R.N = P.ringN[j];
    R.mcut = P.mcut[j];
    R.shifted = P.shifted[j];
    R.start = (r > j) ? P.npix - R.N - P.start[j] : P.start[j];
    R.weight = 1.0;
    if (use_w) R.weight = w ? w[r] : 4.0 * 3.14159265358979323846 / (double)P.npix;
    return R;
}

// ------------------------------------------------------------------ direct kernels (short rings)
template <typename T>
__global__ void __launch_bounds__(FFT_THREADS) ring_direct_analysis_kernel(DevPlan P, const int* __restrict__ rings,
                                                                          const T* __restrict__ map,
                                                                          const double* __restrict__ w, int use_w) {
    using T2 = typename V2<T>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int r = rings[blockIdx.x], ch = blockIdx.y;
    const RingRef R = ring_ref(P, r, w, use_w);
    const int N = R.N;
    T2* tw = reinterpret_cast<T2*>(smem_raw);
    T* p = reinterpret_cast<T*>(tw + N);
    const T* src = map + (size_t)ch * P.npix + R.start;
    for (int x = threadIdx.x; x < N; x += blockDim.x) {
        p[x] = src[x];
        T c, s;
        cispi_ratio(2LL * x, N, (T)-1, c, s);
        tw[x].x = c;
        tw[x].y = s;
    }
    __syncthreads();
    T2* dst = reinterpret_cast<T2*>(P.spectra) + ((size_t)ch * P.nrings + r) * P.mstride;
    for (int m = threadIdx.x; m <= R.mcut; m += blockDim.x) {
        const int step = m % N;
        int idx = 0;
        T ar = 0, ai = 0;
        for (int x = 0; x < N; ++x) {
            ar = fma(p[x], tw[idx].x, ar);
            ai = fma(p[x], tw[idx].y, ai);
            idx += step;
            if (idx >= N) idx -= N;
        }
        T c = 1, s = 0;
        if (R.shifted) cispi_ratio((long long)(m % (2 * N)), N, (T)-1, c, s);
        const T wt = (T)R.weight;
        T2 o;
        o.x = wt * (ar * c - ai * s);
        o.y = wt * (ar * s + ai * c);
        dst[m] = o;
    }
}

template <typename T>
__global__ void __launch_bounds__(FFT_THREADS) ring_direct_synthesis_kernel(DevPlan P, const int* __restrict__ rings,
                                                                           T* __restrict__ map,
                                                                           const double* __restrict__ w, int use_w) {
    using T2 = typename V2<T>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int r = rings[blockIdx.x], ch = blockIdx.y;
    const RingRef R = ring_ref(P, r, w, use_w);
    const int N = R.N;
    T2* tw = reinterpret_cast<T2*>(smem_raw);
    T2* G = tw + N;
    const T2* src = reinterpret_cast<const T2*>(P.spectra) + ((size_t)ch * P.nrings + r) * P.mstride;
    for (int x = threadIdx.x; x < N; x += blockDim.x) {
        T c, s;
        cispi_ratio(2LL * x, N, (T)1, c, s);
        tw[x].x = c;
        tw[x].y = s;
    }
    for (int m = threadIdx.x; m <= R.mcut; m += blockDim.x) {
        T2 g = src[m];
        if (R.shifted) {
            T c, s;
            cispi_ratio((long long)(m % (2 * N)), N, (T)1, c, s);
            const T gr = g.x * c - g.y * s, gi = g.x * s + g.y * c;
            g.x = gr;
            g.y = gi;
        }
        G[m] = g;
    }
    __syncthreads();
    T* dst = map + (size_t)ch * P.npix + R.start;
    for (int x = threadIdx.x; x < N; x += blockDim.x) {
        T acc = 0;
        int idx = 0;
        for (int m = 1; m <= R.mcut; ++m) {
            idx += x;
            if (idx >= N) idx -= N;
            acc = fma(G[m].x, tw[idx].x, acc);
            acc = fma(-G[m].y, tw[idx].y, acc);
        }
        dst[x] = (T)R.weight * (G[0].x + 2 * acc);
    }
}

// ------------------------------------------------------------------ planning
bool fft_supported(int nside, cuhpx_dtype_t dt) {
    (void)dt;
    return 4 * nside <= DIRECT_MAX_N;
}

size_t plan_fft_tables(HostPlan& hp, char* base, bool build, cudaStream_t st, cudaError_t* err) {
    const DevPlan& d = hp.d;
    hp.rings_direct.clear();
    hp.rings_pow2.clear();
    hp.rings_blue.clear();
    for (int r = 0; r < d.nrings; ++r) hp.rings_direct.push_back(r);
    size_t o = 0;
    auto take = [&](size_t bytes) {
        size_t r = o;
        o = (o + bytes + 255) / 256 * 256;
        return r;
    };
    const size_t off_direct = take(sizeof(int) * hp.rings_direct.size());
    if (build) {
        hp.d_rings_direct = (int*)(base + off_direct);
        *err = cudaMemcpyAsync(hp.d_rings_direct, hp.rings_direct.data(), sizeof(int) * hp.rings_direct.size(),
                               cudaMemcpyHostToDevice, st);
        if (*err == cudaSuccess) *err = cudaStreamSynchronize(st);
    }
    return o;
}

// ------------------------------------------------------------------ launchers
template <typename T>
static cudaError_t run_fft_analysis(const HostPlan& hp, const void* d_map, const double* d_w, int use_w,
                                    cudaStream_t st) {
    const DevPlan& P = hp.d;
    if (!hp.rings_direct.empty()) {
        dim3 grid((unsigned)hp.rings_direct.size(), P.batch);
        const size_t smem = (size_t)DIRECT_MAX_N * 3 * sizeof(T);
        ring_direct_analysis_kernel<T><<<grid, FFT_THREADS, smem, st>>>(P, hp.d_rings_direct, (const T*)d_map, d_w, use_w);
    }
    return cudaGetLastError();
}

template <typename T>
static cudaError_t run_fft_synthesis(const HostPlan& hp, void* d_map, const double* d_w, int use_w, cudaStream_t st) {
    const DevPlan& P = hp.d;
    if (!hp.rings_direct.empty()) {
        dim3 grid((unsigned)hp.rings_direct.size(), P.batch);
        const size_t smem = ((size_t)DIRECT_MAX_N + P.mstride) * 2 * sizeof(T);
        ring_direct_synthesis_kernel<T><<<grid, FFT_THREADS, smem, st>>>(P, hp.d_rings_direct, (T*)d_map, d_w, use_w);
    }
    return cudaGetLastError();
}

cudaError_t launch_fft_analysis(const HostPlan& hp, const void* d_map, const double* d_w, int use_w, cudaStream_t st) {
    return hp.dtype == CUHPX_F64 ? run_fft_analysis<double>(hp, d_map, d_w, use_w, st)
                                 : run_fft_analysis<float>(hp, d_map, d_w, use_w, st);
}

cudaError_t launch_fft_synthesis(const HostPlan& hp, void* d_map, const double* d_w, int use_w, cudaStream_t st) {
    return hp.dtype == CUHPX_F64 ? run_fft_synthesis<double>(hp, d_map, d_w, use_w, st)
                                 : run_fft_synthesis<float>(hp, d_map, d_w, use_w, st);
}

}  // namespace cuhpx

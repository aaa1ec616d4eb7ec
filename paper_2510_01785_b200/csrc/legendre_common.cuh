// Pieces shared by the Legendre-stage kernels (legendre.cu: CUDA-core kernels; legendre_tc.cu: tcgen05 kernels):
// exponent windows of the scaled recurrence, the seed lambda_mm (Eq. 15), kernel arguments.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

#include "cuhpx_internal.h"

namespace cuhpx {

template <typename T> struct Vec2;
template <> struct Vec2<float> { using type = float2; };
template <> struct Vec2<double> { using type = double2; };

// Exponent windows of the scaled recurrence.  true lambda = val * 2^(K * sc), sc <= 0.  A ring is "inactive"
// while sc < 0; then |true lambda| < 2^(THR + 56 - K): 2^-200 (fp64) / 2^-44 (fp32 outputs), i.e. it cannot
// change the result.  56 = log2 of the largest growth over the 8 steps between two checks.
template <typename T> struct ScaleCfg;
template <> struct ScaleCfg<double> { static constexpr int THR = 256, K = 512; };
template <> struct ScaleCfg<float> { static constexpr int THR = 60, K = 160; };
__host__ __device__ constexpr double pow2c(int e) {
    double v = 1.0;
    for (int i = 0; i < (e < 0 ? -e : e); ++i) v = e < 0 ? v * 0.5 : v * 2.0;
    return v;
}
constexpr int CHECK_EVERY = 8;  // l steps between rescale checks (must divide CT and be a multiple of LT)

// log2|lambda_mm(theta_j)| = pref[m] + m log2 sin(theta_j), evaluated in double-double so that the seed is
// good to ~1e-16 relative even when the exponent is in the thousands.
template <typename T>
__device__ __forceinline__ void lambda_seed(int m, double pref_hi, double pref_lo, double ls_hi, double ls_lo,
                                            double& val, int& sc) {
    const double dm = (double)m;
    const double p = dm * ls_hi;
    const double pe = fma(dm, ls_hi, -p);
    const double s = p + pref_hi;
    const double bb = s - p;
    const double se = (p - (s - bb)) + (pref_hi - bb);
    const double lo = pe + se + fma(dm, ls_lo, pref_lo);
    const double n = rint(s + lo);
    const double f = (s - n) + lo;
    const double mant = exp2(f);
    int ni = (int)fmax(n, -2.0e9);
    sc = 0;
    constexpr int THR = ScaleCfg<T>::THR, K = ScaleCfg<T>::K;
    if (ni < THR - K) {
        // floor((ni - THR) / K) + 1, written for negative numerators
        const int num = ni - THR;
        const int fl = -((-num + K - 1) / K);
        sc = fl + 1;
        ni -= K * sc;
    }
    val = scalbn(mant, ni);
    if (m & 1) val = -val;
}

struct LegArgs {
    DevPlan p;
    const void* in;  // analysis: unused (spectra from plan); synthesis: alm
    void* out;       // analysis: alm or partial; synthesis: unused
    int adjoint;
    int to_partial;  // analysis: write [chunk][batch][nalm] partial sums
};

// launchers of the tcgen05 kernels (legendre_tc.cu); each returns cudaErrorNotSupported when the shape is not served
cudaError_t launch_legendre_synthesis_tc(const HostPlan& hp, const DevPlan& P, const void* d_alm, int adjoint, cudaStream_t st);

}  // namespace cuhpx

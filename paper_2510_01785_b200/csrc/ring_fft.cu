// FFT stage of the HEALPix SHT: per-ring real DFT in longitude fused with the
// phi0 phase twist and the m-aliasing rule (m mod N_i) of Eq. 24 / Eq. 26.
//   analysis : F_m(i) = w_i exp(-i m phi0_i) X~_i[m mod N_i],  X_i[k] = sum_x p_x exp(-2 pi i k x / N_i)   (Eq. 13)
//   synthesis: p_x = Re G_0 + 2 sum_{m>=1} Re(G_m exp(+i m (phi0_i + 2 pi x / N_i)))                       (Eq. 24)
// Three kernel families, chosen per ring length N:
//   direct   : O(N m_cut) sums for N <= 256 (the first 64 rings of each cap; negligible work)
//   pow2     : N = 2^k (all belt rings, cap rings with i a power of two): real FFT of length N as one complex
//              block FFT of length N/2 held in registers (block_fft.cuh), Hermitian unpack fused with the twist
//   bluestein: the other cap rings, N = 4 i: chirp-z (Eq. 17-23).  Unlike the paper's uniform chirp
//              length + batched cuFFT, each ring uses its own minimal power-of-two length M >= 2i - 1 and
//              stays inside one SM: the packed complex sequence of length 2 i is split into its even and odd
//              halves (two length-i chirp-z transforms), each = chirp multiply -> FFT_M -> filter -> IFFT_M ->
//              chirp multiply, all in registers/shared memory; the filter spectra are precomputed per i.
// One CTA per (ring, channel); rings are read and spectra written exactly once, coalesced.
#include <cuda_runtime.h>
#include <math.h>
#include <string.h>

#include <algorithm>
#include <mutex>
#include <vector>

#include "block_fft.cuh"
#include "cuhpx_internal.h"

namespace cuhpx {

constexpr int DIRECT_MAX_N = 256;
constexpr int FFT_THREADS = 256;  // direct kernels
constexpr int MIN_LOG = 7, MAX_LOG = 13;  // LOG 7: the belt rings of nside 64 (N = 256) as one-warp FFTs

// exp(sign * i * pi * num / den) from exact integers (num already reduced mod 2 den); direct kernels only
__device__ __forceinline__ void cispi_ratio(long long num, long long den, double sign, double& c, double& s) {
    sincospi((double)num / (double)den, &s, &c);
    s *= sign;
}
__device__ __forceinline__ void cispi_ratio(long long num, long long den, float sign, float& c, float& s) {
    sincospif((float)num / (float)den, &s, &c);  // num < 2 den <= 512: exact integers, one rounding
    s *= sign;
}

// One work item of an FFT-stage launch: everything a CTA needs to know about its ring, in one 32-byte record
// (built per plan on the host; replaces four dependent table look-ups).
struct __align__(16) RingInfo {
    long long start;  // RING index of the ring's first pixel
    int N;            // pixels in the ring
    int mcut;         // largest order kept on this ring
    int shifted;      // 1: phi0 = pi / N, 0: phi0 = 0
    int r;            // 0-based ring number, north to south
    int pad0, pad1;
};
static_assert(sizeof(RingInfo) == 32, "RingInfo layout");

__device__ __forceinline__ RingInfo load_info(const RingInfo* __restrict__ info, int idx) {
    const int4 a = __ldg(reinterpret_cast<const int4*>(info + idx));
    const int4 b = __ldg(reinterpret_cast<const int4*>(info + idx) + 1);
    RingInfo R;
    R.start = (long long)(((unsigned long long)(unsigned)a.y << 32) | (unsigned)a.x);
    R.N = a.z;
    R.mcut = a.w;
    R.shifted = b.x;
    R.r = b.y;
    return R;
}

__device__ __forceinline__ double ring_weight(const DevPlan& P, const RingInfo& R, const double* __restrict__ w, int use_w) {
    if (!use_w) return 1.0;
    if (w) return __ldg(w + R.r);
    return P.defw ? __ldg(P.defw + R.r) : 4.0 * 3.14159265358979323846 / (double)P.npix;
}

// Ask the memory system to bring `bytes` at `ptr` into L2 (no register or shared-memory destination): issued
// for the work item the SM will run next, so its HBM traffic overlaps the current item's arithmetic.
__device__ __forceinline__ void prefetch_l2(const void* ptr, unsigned bytes) {
    constexpr unsigned CHUNK = 16384;
    const char* p = reinterpret_cast<const char*>(ptr);
    for (unsigned o = (threadIdx.x & 31) * CHUNK; o < bytes; o += 32 * CHUNK) {
        const unsigned n = min(CHUNK, bytes - o) & ~15u;
        if (n) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p + o), "r"(n) : "memory");
    }
}

struct FftTables {
    const void* tw;  // complex<T>[twlen] = exp(-2 pi i k / twlen)
    int twlen;
    const void* filt;             // Bluestein filter spectra, register order, concatenated
    const long long* filt_offset; // [nside] offset (complex units) for cap ring i, -1 if none
    int pf;                       // prefetch distance in work items (CTAs resident on the GPU at once)
};

// work item of this CTA and L2 prefetch of the item `pf` launches ahead (grid = (items, channels), x fastest)
template <typename T, bool ANALYSIS>
__device__ __forceinline__ RingInfo begin_item(const DevPlan& P, const RingInfo* __restrict__ info, const T* map, int pf) {
    const RingInfo R = load_info(info, blockIdx.x);
    if (threadIdx.x < 32 && pf > 0) {
        const long long lin = (long long)blockIdx.y * gridDim.x + blockIdx.x + pf;
        if (lin < (long long)gridDim.x * gridDim.y) {
            const int nx = (int)(lin % gridDim.x), nch = (int)(lin / gridDim.x);
            const RingInfo Rn = load_info(info, nx);
            if (ANALYSIS) {
                prefetch_l2(map + (size_t)nch * P.npix + Rn.start, (unsigned)(Rn.N * sizeof(T)));
            } else {
                using T2 = typename V2<T>::type;
                const T2* row = reinterpret_cast<const T2*>(P.spectra) + ((size_t)nch * P.nrings + Rn.r) * P.mstride;
                prefetch_l2(row, (unsigned)(((Rn.mcut + 1) * sizeof(T2) + 15) & ~15u));
            }
        }
    }
    return R;
}

// Bluestein kernels: the filter spectrum of the ring size the SM will see `pf` items ahead, brought into L2 as well (it is
// first touched in the middle of a work item, between the forward and the inverse transform, where every warp of the CTA
// waits for it; north and south ring of one size are neighbours in the work list, so every other item finds it anyway)
template <typename T>
__device__ __forceinline__ void prefetch_filter(const RingInfo* __restrict__ info, const FftTables& tabs, int m_len) {
    if (threadIdx.x < 32 && tabs.pf > 0) {
        const long long lin = (long long)blockIdx.y * gridDim.x + blockIdx.x + tabs.pf;
        if (lin < (long long)gridDim.x * gridDim.y) {
            const RingInfo Rn = load_info(info, (int)(lin % gridDim.x));
            using T2 = typename V2<T>::type;
            const T2* f = reinterpret_cast<const T2*>(tabs.filt) + __ldg(tabs.filt_offset + (Rn.N >> 2));
            prefetch_l2(f, (unsigned)(m_len * sizeof(T2)));
        }
    }
}

// ------------------------------------------------------------------ direct kernels (short rings)
template <typename T>
__global__ void __launch_bounds__(FFT_THREADS) ring_direct_analysis_kernel(DevPlan P, const RingInfo* __restrict__ info,
                                                                          const T* __restrict__ map,
                                                                          const double* __restrict__ w, int use_w) {
    if (!ws_ok(P)) return;
    using T2 = typename V2<T>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int ch = blockIdx.y;
    const RingInfo R = load_info(info, blockIdx.x);
    const int N = R.N, r = R.r;
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
    const T wt = (T)ring_weight(P, R, w, use_w);
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
        T2 o;
        o.x = wt * (ar * c - ai * s);
        o.y = wt * (ar * s + ai * c);
        dst[m] = o;
    }
}

template <typename T>
__global__ void __launch_bounds__(FFT_THREADS) ring_direct_synthesis_kernel(DevPlan P, const RingInfo* __restrict__ info,
                                                                           T* __restrict__ map,
                                                                           const double* __restrict__ w, int use_w) {
    if (!ws_ok(P)) return;
    using T2 = typename V2<T>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int ch = blockIdx.y;
    const RingInfo R = load_info(info, blockIdx.x);
    const int N = R.N, r = R.r;
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
    const T wt = (T)ring_weight(P, R, w, use_w);
    for (int x = threadIdx.x; x < N; x += blockDim.x) {
        T acc = 0;
        int idx = 0;
        for (int m = 1; m <= R.mcut; ++m) {
            idx += x;
            if (idx >= N) idx -= N;
            acc = fma(G[m].x, tw[idx].x, acc);
            acc = fma(-G[m].y, tw[idx].y, acc);
        }
        dst[x] = wt * (G[0].x + 2 * acc);
    }
}

// ------------------------------------------------------------------ direct kernels, channel-blocked (batched maps)
// With many channels (BASELINE configs[2]: nside 64, 256 channels -- every ring is a "short" ring) the direct sums
// are the whole FFT stage.  One CTA = (ring, CB channels): a twiddle is fetched once per (m, x) and used for CB
// channels (2 CB FMAs per shared-memory twiddle instead of 2), the ring data of the CB channels sits in shared
// memory as [x][CB] so one broadcast LDS.128 feeds 4 channels.
constexpr int DIRECT_CB_THREADS = 128;

template <typename T, int CB>
__global__ void __launch_bounds__(DIRECT_CB_THREADS) ring_direct_analysis_cb_kernel(DevPlan P, const RingInfo* __restrict__ info,
                                                                                   const T* __restrict__ map,
                                                                                   const double* __restrict__ w, int use_w) {
    if (!ws_ok(P)) return;
    using T2 = typename V2<T>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int ch0 = blockIdx.y * CB;
    const RingInfo R = load_info(info, blockIdx.x);
    const int N = R.N, r = R.r, tid = threadIdx.x;
    T2* tw = reinterpret_cast<T2*>(smem_raw);
    T* p = reinterpret_cast<T*>(tw + N);  // [x][CB]
    for (int x = tid; x < N; x += DIRECT_CB_THREADS) {
        T c, s;
        cispi_ratio(2LL * x, N, (T)-1, c, s);
        tw[x].x = c;
        tw[x].y = s;
    }
    for (int e = tid; e < N * CB; e += DIRECT_CB_THREADS) {
        const int c = e / N, x = e - c * N, ch = ch0 + c;
        p[x * CB + c] = ch < P.batch ? map[(size_t)ch * P.npix + R.start + x] : (T)0;
    }
    __syncthreads();
    const T wt = (T)ring_weight(P, R, w, use_w);
    for (int m = tid; m <= R.mcut; m += DIRECT_CB_THREADS) {
        const int step = m % N;
        int idx = 0;
        T ar[CB], ai[CB];
#pragma unroll
        for (int c = 0; c < CB; ++c) ar[c] = ai[c] = 0;
        for (int x = 0; x < N; ++x) {
            const T2 t = tw[idx];
            T pv[CB];
#pragma unroll
            for (int c = 0; c < CB; c += 4 / (sizeof(T) / 4)) {  // 16-byte broadcast loads
                if (sizeof(T) == 4) {
                    const float4 v = *reinterpret_cast<const float4*>(&p[x * CB + c]);
                    pv[c] = v.x; pv[c + 1] = v.y; pv[c + 2] = v.z; pv[c + 3] = v.w;
                } else {
                    const double2 v = *reinterpret_cast<const double2*>(&p[x * CB + c]);
                    pv[c] = v.x; pv[c + 1] = v.y;
                }
            }
#pragma unroll
            for (int c = 0; c < CB; ++c) {
                ar[c] = fma(pv[c], t.x, ar[c]);
                ai[c] = fma(pv[c], t.y, ai[c]);
            }
            idx += step;
            if (idx >= N) idx -= N;
        }
        T c = 1, s = 0;
        if (R.shifted) cispi_ratio((long long)(m % (2 * N)), N, (T)-1, c, s);
#pragma unroll
        for (int k = 0; k < CB; ++k) {
            const int ch = ch0 + k;
            if (ch < P.batch) {
                T2 o;
                o.x = wt * (ar[k] * c - ai[k] * s);
                o.y = wt * (ar[k] * s + ai[k] * c);
                (reinterpret_cast<T2*>(P.spectra) + ((size_t)ch * P.nrings + r) * P.mstride)[m] = o;
            }
        }
    }
}

template <typename T, int CB>
__global__ void __launch_bounds__(DIRECT_CB_THREADS) ring_direct_synthesis_cb_kernel(DevPlan P, const RingInfo* __restrict__ info,
                                                                                    T* __restrict__ map,
                                                                                    const double* __restrict__ w, int use_w) {
    if (!ws_ok(P)) return;
    using T2 = typename V2<T>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int ch0 = blockIdx.y * CB;
    const RingInfo R = load_info(info, blockIdx.x);
    const int N = R.N, r = R.r, tid = threadIdx.x, nm = R.mcut + 1;
    T2* tw = reinterpret_cast<T2*>(smem_raw);
    T2* G = tw + N;  // [m][CB], already twisted by exp(+i m phi0)
    for (int x = tid; x < N; x += DIRECT_CB_THREADS) {
        T c, s;
        cispi_ratio(2LL * x, N, (T)1, c, s);
        tw[x].x = c;
        tw[x].y = s;
    }
    for (int e = tid; e < nm * CB; e += DIRECT_CB_THREADS) {
        const int k = e / nm, m = e - k * nm, ch = ch0 + k;
        T2 g;
        g.x = g.y = 0;
        if (ch < P.batch) g = (reinterpret_cast<const T2*>(P.spectra) + ((size_t)ch * P.nrings + r) * P.mstride)[m];
        if (m == 0) g.y = 0;  // Im G_0 is ignored
        if (R.shifted) {
            T c, s;
            cispi_ratio((long long)(m % (2 * N)), N, (T)1, c, s);
            const T gr = g.x * c - g.y * s, gi = g.x * s + g.y * c;
            g.x = gr;
            g.y = gi;
        }
        G[m * CB + k] = g;
    }
    __syncthreads();
    const T wt = (T)ring_weight(P, R, w, use_w);
    for (int x = tid; x < N; x += DIRECT_CB_THREADS) {
        T acc[CB];
#pragma unroll
        for (int k = 0; k < CB; ++k) acc[k] = 0;
        int idx = 0;
        for (int m = 1; m < nm; ++m) {
            idx += x;
            if (idx >= N) idx -= N;
            const T2 t = tw[idx];
#pragma unroll
            for (int k = 0; k < CB; ++k) {
                const T2 g = G[m * CB + k];
                acc[k] = fma(g.x, t.x, acc[k]);
                acc[k] = fma(-g.y, t.y, acc[k]);
            }
        }
#pragma unroll
        for (int k = 0; k < CB; ++k) {
            const int ch = ch0 + k;
            if (ch < P.batch) map[(size_t)ch * P.npix + R.start + x] = wt * (G[k].x + 2 * acc[k]);
        }
    }
}

// ------------------------------------------------------------------ shared pieces of the FFT kernels
// Every phase factor of a ring of N pixels is a power of omega = exp(-2 pi i / Q), Q = 2 N:
//   twist exp(-i m phi0) = omega^m (phi0 = pi / N),  W_N^k = omega^(2 k),  W_{N/2}^k = omega^(4 k).
// `rt` is the shared-memory root table of order Q (block_fft.cuh).
template <bool POW2> __device__ __forceinline__ int mod_q(int m, int Q) { return POW2 ? (m & (Q - 1)) : (m % Q); }

// Folded half spectrum H[k], k = 0..n (n = N/2), of the synthesis input:
//   c_m = G_m exp(+i m phi0);  0 < k < n: H[k] = sum_{m = k (N)} c_m + sum_{m = -k (N)} conj(c_m);
//   k in {0, n}: H[k] = sum_{m = k (N)} (m == 0 ? Re c_0 : 2 Re c_m)
template <typename T, bool POW2>
__device__ __forceinline__ void folded_H(const typename V2<T>::type* __restrict__ G, int k, int N, int mcut, int shifted,
                                         const Roots<T>& rt, T& hr, T& hi) {
    using T2 = typename V2<T>::type;
    const int n = N >> 1;
    hr = 0;
    hi = 0;
    auto cm = [&](int m, T& cr, T& ci) {
        const T2 g = G[m];
        if (shifted) {
            T c, s;
            rt.template get<+1>(mod_q<POW2>(m, 2 * N), c, s);
            cr = g.x * c - g.y * s;
            ci = g.x * s + g.y * c;
        } else {
            cr = g.x;
            ci = g.y;
        }
    };
    if (k == 0 || k == n) {
        for (int m = k; m <= mcut; m += N) {
            T cr, ci;
            cm(m, cr, ci);
            hr += (m == 0) ? cr : 2 * cr;
        }
    } else {
        for (int m = k; m <= mcut; m += N) {
            T cr, ci;
            cm(m, cr, ci);
            hr += cr;
            hi += ci;
        }
        for (int m = N - k; m <= mcut; m += N) {
            T cr, ci;
            cm(m, cr, ci);
            hr += cr;
            hi -= ci;
        }
    }
}

// Packed inverse-real-FFT input: Y[k] = conj(Zs[k]), Zs[k] = E' + i O', E' = H[k] + conj H[n-k],
// O' = (H[k] - conj H[n-k]) exp(+2 pi i k / N); the ring is then x[2t] = Re D[t], x[2t+1] = -Im D[t], D = DFT_n(Y).
template <typename T, bool POW2>
__device__ __forceinline__ void synth_packed_input(const typename V2<T>::type* __restrict__ G, int k, int N, int mcut,
                                                   int shifted, const Roots<T>& rt, T& yr, T& yi) {
    using T2 = typename V2<T>::type;
    const int n = N >> 1;
    T ar, ai, br, bi, c, s;
    if (mcut < n) {
        // no order reaches the Nyquist bin: H[k] = G_k e^{i k phi0} for k <= mcut, else 0.  With p = e^{i pi k / N}:
        // twist of bin k is p, of bin n - k is i conj(p), and e^{2 pi i k / N} = p^2: one root per element.
        T pc, ps;
        rt.template get<+1>(k, pc, ps);
        T2 a, b;
        a.x = a.y = b.x = b.y = 0;
        if (k <= mcut) a = G[k];
        if (n - k <= mcut) b = G[n - k];
        if (k == 0) a.y = 0;  // Im G_0 is ignored
        if (shifted) {
            ar = a.x * pc - a.y * ps;
            ai = a.x * ps + a.y * pc;
            br = b.x * ps - b.y * pc;  // b * (ps + i pc)
            bi = b.x * pc + b.y * ps;
        } else {
            ar = a.x; ai = a.y; br = b.x; bi = b.y;
        }
        c = pc * pc - ps * ps;
        s = 2 * pc * ps;
    } else {
        folded_H<T, POW2>(G, k, N, mcut, shifted, rt, ar, ai);
        folded_H<T, POW2>(G, n - k, N, mcut, shifted, rt, br, bi);
        rt.template get<+1>(2 * k, c, s);
    }
    bi = -bi;  // conj H[n-k]
    const T er = ar + br, ei = ai + bi;
    const T dr = ar - br, di = ai - bi;
    const T orr = dr * c - di * s, oi = dr * s + di * c;
    // Zs = E' + i O' = (er - oi) + i (ei + orr);  Y = conj
    yr = er - oi;
    yi = -(ei + orr);
}

// Hermitian unpack of the packed analysis FFT + twist: given Z[kk mod n] and Z[(n-kk) mod n] returns
// F_m = weight * exp(-i m phi0) * X~[m mod N]  (k = m mod N, kk = min(k, N - k), cj = k > n)
template <typename T, bool POW2>
__device__ __forceinline__ typename V2<T>::type analysis_unpack(T z1r, T z1i, T z2r, T z2i, int m, int kk, bool cj, int N,
                                                                 int shifted, T wt, const Roots<T>& rt) {
    const T er = (T)0.5 * (z1r + z2r), ei = (T)0.5 * (z1i - z2i);
    const T dr = (T)0.5 * (z1r - z2r), di = (T)0.5 * (z1i + z2i);
    // O = -i D = (di, -dr);  X = E + W_N^kk O.  Unaliased (kk == m): W_N^kk = omega^(2 m) is the square of the twist.
    T pc, ps, c, s;
    const bool plain = (kk == m);
    rt.template get<-1>(plain ? m : mod_q<POW2>(m, 2 * N), pc, ps);  // twist omega^m
    if (plain) {
        c = pc * pc - ps * ps;
        s = 2 * pc * ps;
    } else {
        rt.template get<-1>(2 * kk, c, s);
    }
    T xr = er + (c * di + s * dr);
    T xi = ei + (s * di - c * dr);
    if (cj) xi = -xi;
    if (shifted) {
        const T tr = xr * pc - xi * ps, ti = xr * ps + xi * pc;
        xr = tr;
        xi = ti;
    }
    typename V2<T>::type o;
    o.x = wt * xr;
    o.y = wt * xi;
    return o;
}

// Hermitian unpack of TWO outputs at once: the bins k and n - k (n = N / 2, 0 <= k <= n / 2) of the packed analysis FFT
// share E = (Z[k] + conj Z[n-k]) / 2 and O = -i (Z[k] - conj Z[n-k]) / 2, and W_N^(n-k) = -conj(W_N^k):
//   X[k] = E + W_N^k O,   X[n-k] = conj(E - W_N^k O);   twists: omega^k and omega^(n-k) = -i conj(omega^k).
// One root look-up and ~29 flops for two outputs (the one-at-a-time unpack: two look-ups and ~30 flops per output).
// z1 = Z[k], z2 = Z[(n - k) mod n]; (pc, ps) = omega^k = exp(-i pi k / N); h = weight / 2.  Valid for k = 0 (f2 = X[n],
// the Nyquist bin) and k = n / 2 (f1 = f2).
template <typename T>
__device__ __forceinline__ void analysis_unpack_pair(T z1r, T z1i, T z2r, T z2i, T pc, T ps, int shifted, T h,
                                                     typename V2<T>::type& f1, typename V2<T>::type& f2) {
    const T er = z1r + z2r, ei = z1i - z2i;      // 2 E
    const T orr = z1i + z2i, oi = z2r - z1r;     // 2 O = -i (z1 - conj z2)
    const T wc = pc * pc - ps * ps, ws = 2 * pc * ps;  // W_N^k = omega^(2 k)
    const T tr = wc * orr - ws * oi, ti = wc * oi + ws * orr;
    const T x1r = er + tr, x1i = ei + ti;        // 2 X[k]
    const T x2r = er - tr, x2i = ei - ti;        // 2 conj X[n-k]
    if (shifted) {
        const T hc = h * pc, hs = h * ps;
        f1.x = x1r * hc - x1i * hs;
        f1.y = x1r * hs + x1i * hc;
        const T ur = x2r * hc - x2i * hs, ui = x2r * hs + x2i * hc;  // h omega^k (2 conj X[n-k])
        f2.x = -ui;  // -i conj(u)
        f2.y = -ur;
    } else {
        f1.x = h * x1r;
        f1.y = h * x1i;
        f2.x = h * x2r;
        f2.y = -h * x2i;
    }
}

// Resident CTAs per SM the register allocation aims for: 16 points per thread are 64 (fp64) / 32 (fp32) data
// registers, so fp64 kernels get 128 registers per thread and fp32 pow2 kernels 64.
template <typename T, int LOG> struct MinBlocks {
    static constexpr int NT = FftPlan<LOG>::NT;
    static constexpr int value = (sizeof(T) == 4 ? 1024 : 512) / NT > 16 ? 16 : (sizeof(T) == 4 ? 1024 : 512) / NT;
    static constexpr int blue = (sizeof(T) == 4 ? 768 : 512) / NT;  // fp32: 80 registers, 6 CTAs of 128 threads per SM (measured best of 4 / 6 / 8)
};

// ------------------------------------------------------------------ power-of-two rings
// shared memory: [exchange buffer of n complex][root table of order Q = 2 N = 4 n]
template <typename T, int LOGN>
__global__ void __launch_bounds__(FftPlan<LOGN>::NT, MinBlocks<T, LOGN>::value) ring_pow2_analysis_kernel(DevPlan P, const RingInfo* __restrict__ info,
                                                                               const T* __restrict__ map,
                                                                               const double* __restrict__ w, int use_w,
                                                                               FftTables tabs) {
    if (!ws_ok(P)) return;
    using F = BlockFFT<T, LOGN, LOGN + 2>;
    using T2 = typename V2<T>::type;
    constexpr int n = F::N, N = 2 * n, Q = 2 * N, E = F::E, NT = F::NT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Xchg<T> xs(smem_raw, n);
    T2* rbase = reinterpret_cast<T2*>(smem_raw + Xchg<T>::bytes(n));
    const int tid = threadIdx.x;
    const int ch = blockIdx.y;
    const RingInfo R = begin_item<T, true>(P, info, map, tabs.pf);
    const T2* src = reinterpret_cast<const T2*>(map + (size_t)ch * P.npix + R.start);
    T re[E], im[E];
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const T2 z = src[F::index0(tid, e)];
        re[e] = z.x;
        im[e] = z.y;
    }
    fill_roots_pow2<T>(rbase, Q, reinterpret_cast<const T2*>(tabs.tw), tabs.twlen, tid, NT);
    const T wt = (T)ring_weight(P, R, w, use_w);
    __syncthreads();
    const Roots<T> rt(rbase);
    F::forward(re, im, xs, rt, tid);
    F::store_natural(re, im, xs, tid);
    __syncthreads();
    T2* dst = reinterpret_cast<T2*>(P.spectra) + ((size_t)ch * P.nrings + R.r) * P.mstride;
    const T h = (T)0.5 * wt;
    const int mcut = R.mcut;
#pragma unroll 2
    for (int k = tid; k <= n / 2; k += NT) {  // orders k and n - k together
        if (k > mcut) break;
        T z1r, z1i, z2r, z2i, pc, ps;
        xs.ld(k, z1r, z1i);
        xs.ld((n - k) & (n - 1), z2r, z2i);
        rt.template get<-1>(k, pc, ps);
        T2 f1, f2;
        analysis_unpack_pair<T>(z1r, z1i, z2r, z2i, pc, ps, R.shifted, h, f1, f2);
        dst[k] = f1;
        if (n - k <= mcut && 2 * k != n) dst[n - k] = f2;
    }
    for (int m = n + 1 + tid; m <= mcut; m += NT) {  // aliased orders (lmax beyond the ring's Nyquist frequency)
        const int k = m & (N - 1);
        const bool cj = k > n;
        const int kk = cj ? N - k : k;
        T z1r, z1i, z2r, z2i;
        xs.ld(kk & (n - 1), z1r, z1i);
        xs.ld((n - kk) & (n - 1), z2r, z2i);
        dst[m] = analysis_unpack<T, true>(z1r, z1i, z2r, z2i, m, kk, cj, N, R.shifted, wt, rt);
    }
}

template <typename T, int LOGN>
__global__ void __launch_bounds__(FftPlan<LOGN>::NT, MinBlocks<T, LOGN>::value) ring_pow2_synthesis_kernel(DevPlan P, const RingInfo* __restrict__ info,
                                                                                T* __restrict__ map,
                                                                                const double* __restrict__ w, int use_w,
                                                                                FftTables tabs) {
    if (!ws_ok(P)) return;
    using F = BlockFFT<T, LOGN, LOGN + 2>;
    using T2 = typename V2<T>::type;
    constexpr int n = F::N, N = 2 * n, Q = 2 * N, E = F::E, NT = F::NT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Xchg<T> xs(smem_raw, n);
    T2* rbase = reinterpret_cast<T2*>(smem_raw + Xchg<T>::bytes(n));
    const int tid = threadIdx.x;
    const int ch = blockIdx.y;
    const RingInfo R = begin_item<T, false>(P, info, map, tabs.pf);
    fill_roots_pow2<T>(rbase, Q, reinterpret_cast<const T2*>(tabs.tw), tabs.twlen, tid, NT);
    const T wt = (T)ring_weight(P, R, w, use_w);
    __syncthreads();
    const Roots<T> rt(rbase);
    const T2* G = reinterpret_cast<const T2*>(P.spectra) + ((size_t)ch * P.nrings + R.r) * P.mstride;
    T re[E], im[E];
#pragma unroll
    for (int e = 0; e < E; ++e)
        synth_packed_input<T, true>(G, F::index0(tid, e), N, R.mcut, R.shifted, rt, re[e], im[e]);
    F::forward(re, im, xs, rt, tid);
    F::store_natural(re, im, xs, tid);
    __syncthreads();
    T2* dst = reinterpret_cast<T2*>(map + (size_t)ch * P.npix + R.start);
#pragma unroll
    for (int t = tid; t < n; t += NT) {
        T a, b;
        xs.ld(t, a, b);
        T2 o;
        o.x = wt * a;
        o.y = -wt * b;
        dst[t] = o;
    }
}

// ------------------------------------------------------------------ long power-of-two rings in halves
// A packed FFT of n = 2 H points whose registers fill a whole SM (fp64, N = 16384: 8192 complex = half of the register
// file, one 512-thread CTA per SM, load / passes / store never overlap) is split with one radix-2 step:
//
// analysis: work item = (ring, parity p of the output bin).  Z[2 k' + p] = FFT_H(y_p)[k'],
//   y_p[j] = (z[j] + (-1)^p z[j + H]) W_n^(p j), formed while loading; the Hermitian partners k and n - k have the same
//   parity, so the unpack stays inside the item.  256 threads, two items resident per SM: one loads or stores while
//   the other computes.  Both items of a ring read the whole ring (the second read comes from L2) and write every
//   other 16-byte bin of the spectra row (the halves of a 32-byte sector meet in L2, microseconds apart).
// synthesis: one CTA of two teams of NT threads; team g transforms the inputs of parity g, Y[2 k' + g] (decimation in
//   time: D[t] = A[t] + W_n^t B[t], D[t + H] = A[t] - W_n^t B[t]); the teams meet only at their own named barriers
//   during the passes, then all threads combine and store whole sectors of the map.
template <typename T, int LOGH>
__global__ void __launch_bounds__(FftPlan<LOGH>::NT, 2) ring_pow2_half_analysis_kernel(DevPlan P, const RingInfo* __restrict__ info,
                                                                                      const T* __restrict__ map,
                                                                                      const double* __restrict__ w, int use_w,
                                                                                      FftTables tabs) {
    if (!ws_ok(P)) return;
    using F = BlockFFT<T, LOGH, LOGH + 3>;
    using T2 = typename V2<T>::type;
    constexpr int H = F::N, n = 2 * H, N = 2 * n, Q = 2 * N, E = F::E, NT = F::NT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Xchg<T> xs(smem_raw, H);
    T2* rbase = reinterpret_cast<T2*>(smem_raw + Xchg<T>::bytes(H));
    const int tid = threadIdx.x;
    const int ch = blockIdx.y;
    const int par = blockIdx.x & 1;
    const RingInfo R = load_info(info, blockIdx.x >> 1);
    const T2* src = reinterpret_cast<const T2*>(map + (size_t)ch * P.npix + R.start);
    T re[E], im[E];
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int j = F::index0(tid, e);
        const T2 a = src[j], b = src[j + H];
        re[e] = par ? a.x - b.x : a.x + b.x;
        im[e] = par ? a.y - b.y : a.y + b.y;
    }
    fill_roots_pow2<T>(rbase, Q, reinterpret_cast<const T2*>(tabs.tw), tabs.twlen, tid, NT);
    const T wt = (T)ring_weight(P, R, w, use_w);
    __syncthreads();
    const Roots<T> rt(rbase);
    if (par) {
        // times W_n^j = omega^(4 j), j = index0(tid, 0) + d_e with d_e a compile-time offset: one look-up per thread,
        // the d_e factors are warp-uniform (broadcast) table entries
        T w0c, w0s;
        rt.template get<-1>(4 * F::index0(tid, 0), w0c, w0s);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int d = F::index0(0, e) - F::index0(0, 0);
            T cc, cs;
            rt.template get<-1>(4 * d, cc, cs);
            const T wc = w0c * cc - w0s * cs, ws = w0c * cs + w0s * cc;
            const T a = re[e], b = im[e];
            re[e] = a * wc - b * ws;
            im[e] = a * ws + b * wc;
        }
    }
    F::forward(re, im, xs, rt, tid);
    F::store_natural(re, im, xs, tid);
    __syncthreads();
    // bins k = 2 k' + par; partner n - k = 2 k'' + par with k'' = (H - k' - par) mod H
    T2* dst = reinterpret_cast<T2*>(P.spectra) + ((size_t)ch * P.nrings + R.r) * P.mstride;
    const T h = (T)0.5 * wt;
    const int mcut = R.mcut;
    const int npairs = par ? H / 2 : H / 2 + 1;
#pragma unroll 2
    for (int kp = tid; kp < npairs; kp += NT) {
        const int k = 2 * kp + par;
        if (k > mcut) break;
        T z1r, z1i, z2r, z2i, pc, ps;
        xs.ld(kp, z1r, z1i);
        xs.ld((H - kp - par) & (H - 1), z2r, z2i);
        rt.template get<-1>(k, pc, ps);
        T2 f1, f2;
        analysis_unpack_pair<T>(z1r, z1i, z2r, z2i, pc, ps, R.shifted, h, f1, f2);
        dst[k] = f1;
        if (n - k <= mcut && 2 * k != n) dst[n - k] = f2;
    }
}

template <typename T, int LOGH>
__global__ void __launch_bounds__(2 * FftPlan<LOGH>::NT, 1) ring_pow2_teams_synthesis_kernel(DevPlan P, const RingInfo* __restrict__ info,
                                                                                            T* __restrict__ map,
                                                                                            const double* __restrict__ w, int use_w,
                                                                                            FftTables tabs) {
    if (!ws_ok(P)) return;
    using F = BlockFFT<T, LOGH, LOGH + 3, 2>;
    using T2 = typename V2<T>::type;
    constexpr int H = F::N, n = 2 * H, N = 2 * n, Q = 2 * N, E = F::E, NT = F::NT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, team = tid / NT, tt = tid % NT;
    const Xchg<T> xa(smem_raw, H), xb(smem_raw + Xchg<T>::bytes(H), H);
    const Xchg<T>& xs = team ? xb : xa;
    T2* rbase = reinterpret_cast<T2*>(smem_raw + 2 * Xchg<T>::bytes(H));
    const int ch = blockIdx.y;
    const RingInfo R = begin_item<T, false>(P, info, map, tabs.pf);
    fill_roots_pow2<T>(rbase, Q, reinterpret_cast<const T2*>(tabs.tw), tabs.twlen, tid, 2 * NT);
    const T wt = (T)ring_weight(P, R, w, use_w);
    __syncthreads();
    const Roots<T> rt(rbase);
    const T2* G = reinterpret_cast<const T2*>(P.spectra) + ((size_t)ch * P.nrings + R.r) * P.mstride;
    T re[E], im[E];
#pragma unroll
    for (int e = 0; e < E; ++e)
        synth_packed_input<T, true>(G, 2 * F::index0(tt, e) + team, N, R.mcut, R.shifted, rt, re[e], im[e]);
    F::forward(re, im, xs, rt, tt);
    F::store_natural(re, im, xs, tt);
    __syncthreads();
    T2* dst = reinterpret_cast<T2*>(map + (size_t)ch * P.npix + R.start);
#pragma unroll 2
    for (int t = tid; t < H; t += 2 * NT) {
        T ar, ai, br, bi, c, s;
        xa.ld(t, ar, ai);
        xb.ld(t, br, bi);
        rt.template get<-1>(4 * t, c, s);  // W_n^t
        const T pr = br * c - bi * s, pi = br * s + bi * c;
        T2 o;
        o.x = wt * (ar + pr);
        o.y = -wt * (ai + pi);
        dst[t] = o;
        o.x = wt * (ar - pr);
        o.y = -wt * (ai - pi);
        dst[t + H] = o;
    }
}

// ------------------------------------------------------------------ Bluestein rings (N = 4 i, i not a power of two)
// shared memory: [exchange buffer of M complex][Ze / De: M/2 + 2 complex][roots of order Q = 8 i][roots of order M]
// chirp c[u] = exp(-i pi u^2 / i) = omega^(4 (u^2 mod 2 i)), omega = exp(-2 pi i / 8 i)   (Eq. 19 P:222 with N -> i)
__device__ __forceinline__ int chirp_index(int u, int twoi, float inv_twoi) {
    const unsigned t = (unsigned)u * (unsigned)u;  // < 2^24: exact in fp32
    const int q = (int)((float)t * inv_twoi);      // floor(t / 2i) +- 1
    int r = (int)t - q * twoi;
    if (r < 0) r += twoi;
    if (r >= twoi) r -= twoi;
    return 4 * r;
}

// One length-i chirp-z transform of the sequence already multiplied by the chirp and zero-padded in registers
// (pass-0 layout): FFT_M -> times filter spectrum -> IFFT_M (Eq. 22).  Result: conv[idx] in registers.
template <typename T, int LOGM>
__device__ __forceinline__ void chirp_convolve(T (&re)[BlockFFT<T, LOGM>::E], T (&im)[BlockFFT<T, LOGM>::E], const Xchg<T>& xs,
                                               const Roots<T>& rtM, const typename V2<T>::type* __restrict__ filt, int tid) {
    using F = BlockFFT<T, LOGM>;
    F::forward(re, im, xs, rtM, tid);
#pragma unroll
    for (int e = 0; e < F::E; ++e) {
        const typename V2<T>::type f = __ldg(filt + e * F::NT + tid);
        const T a = re[e], b = im[e];
        re[e] = a * f.x - b * f.y;
        im[e] = a * f.y + b * f.x;
    }
    F::inverse(re, im, xs, rtM, tid);
}

template <typename T, int LOGM> struct BlueSmem {
    static constexpr int M = 1 << LOGM;
    static constexpr size_t off_z = Xchg<T>::bytes(M);
    static constexpr size_t off_rq = off_z + sizeof(T) * 2 * ((size_t)M / 2 + 2);
    static constexpr size_t off_rm = off_rq + sizeof(T) * 2 * (size_t)roots_len(4 * M + 8);  // Q = 8 i <= 4 M + 8
    static constexpr size_t off_cs = off_rm + sizeof(T) * 2 * (size_t)roots_len(M);
    // fp32 only: the thread's own chirp factors [e][tid] (each is needed 4 times: before / after the convolution of
    // both sub-sequences; ~20 instructions to rebuild, one LDS.64 to reload).  fp64 has no shared memory to spare.
    static constexpr bool KEEP_CHIRP = sizeof(T) == 4 && LOGM <= 12;  // beyond, the table would halve the resident CTAs
    static constexpr size_t total = off_cs + (KEEP_CHIRP ? sizeof(T) * 2 * (size_t)M : 0);
};

template <typename T, int LOGM>
__global__ void __launch_bounds__(FftPlan<LOGM>::NT, MinBlocks<T, LOGM>::blue) ring_blue_analysis_kernel(DevPlan P, const RingInfo* __restrict__ info,
                                                                               const T* __restrict__ map,
                                                                               const double* __restrict__ w, int use_w,
                                                                               FftTables tabs) {
    if (!ws_ok(P)) return;
    using F = BlockFFT<T, LOGM>;
    using T2 = typename V2<T>::type;
    using SM = BlueSmem<T, LOGM>;
    constexpr int M = F::N, E = F::E, NT = F::NT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Xchg<T> xs(smem_raw, M);
    T2* Ze = reinterpret_cast<T2*>(smem_raw + SM::off_z);
    T2* rq = reinterpret_cast<T2*>(smem_raw + SM::off_rq);
    T2* rm = reinterpret_cast<T2*>(smem_raw + SM::off_rm);
    const int tid = threadIdx.x;
    const int ch = blockIdx.y;
    const RingInfo R = begin_item<T, true>(P, info, map, tabs.pf);
    prefetch_filter<T>(info, tabs, M);
    const int N = R.N, i = N >> 2, n = N >> 1, Q = 2 * N;
    const T2* src = reinterpret_cast<const T2*>(map + (size_t)ch * P.npix + R.start);
    const T2* filt = reinterpret_cast<const T2*>(tabs.filt) + __ldg(tabs.filt_offset + i);
    fill_roots_any<T>(rq, Q, tid, NT);
    fill_roots_pow2<T>(rm, M, reinterpret_cast<const T2*>(tabs.tw), tabs.twlen, tid, NT);
    const T wt = (T)ring_weight(P, R, w, use_w);
    const float inv_twoi = 1.0f / (float)(2 * i);
    __syncthreads();
    const Roots<T> rt(rq), rtM(rm);
    T2* cs = reinterpret_cast<T2*>(smem_raw + SM::off_cs) + tid;  // [e * NT]: private to this thread
    if constexpr (SM::KEEP_CHIRP) {
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int u = F::index0(tid, e);
            T2 v;
            v.x = 1;
            v.y = 0;
            if (u < i) rt.template get<-1>(chirp_index(u, 2 * i, inv_twoi), v.x, v.y);
            cs[e * NT] = v;
        }
    }
    T re[E], im[E];
#pragma unroll 1
    for (int sub = 0; sub < 2; ++sub) {
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int u = F::index0(tid, e);
            re[e] = 0;
            im[e] = 0;
            if (u < i) {
                const T2 z = src[2 * u + sub];
                T c, s;
                if constexpr (SM::KEEP_CHIRP) {
                    const T2 v = cs[e * NT];
                    c = v.x;
                    s = v.y;
                } else {
                    rt.template get<-1>(chirp_index(u, 2 * i, inv_twoi), c, s);
                }
                re[e] = z.x * c - z.y * s;
                im[e] = z.x * s + z.y * c;
            }
        }
        chirp_convolve<T, LOGM>(re, im, xs, rtM, filt, tid);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int u = F::index0(tid, e);
            if (u < i) {
                T c, s;
                if constexpr (SM::KEEP_CHIRP) {
                    const T2 v = cs[e * NT];
                    c = v.x;
                    s = v.y;
                } else {
                    rt.template get<-1>(chirp_index(u, 2 * i, inv_twoi), c, s);
                }
                const T vr = re[e] * c - im[e] * s, vi = re[e] * s + im[e] * c;
                if (sub == 0) {
                    T2 v;
                    v.x = vr;
                    v.y = vi;
                    Ze[u] = v;
                } else {  // own pass-0 slot of the exchange buffer: no other thread touches it
                    xs.st(u, vr, vi);
                }
            }
        }
    }
    __syncthreads();
    // Z[q] = Ze[q mod i] + W_n^q Zo[q mod i], q < n = 2 i.  twist = omega^m, W_N^kk = omega^(2 kk),
    // W_n^q = omega^(4 q); without aliasing (m <= n, the common case) kk = m and one root per output suffices.
    T2* dst = reinterpret_cast<T2*>(P.spectra) + ((size_t)ch * P.nrings + R.r) * P.mstride;
    const int mcut = R.mcut;
    const T h = (T)0.5 * wt;
    // orders kk and n - kk together (they share E / O, see analysis_unpack_pair); W_n^(n - kk) = conj(W_n^kk)
#pragma unroll 2
    for (int kk = tid; kk <= i; kk += NT) {
        if (kk > mcut) break;
        T pc, ps;  // omega^kk
        rt.template get<-1>(kk, pc, ps);
        const T w2c = pc * pc - ps * ps, w2s = 2 * pc * ps;        // W_N^kk
        const T w4c = w2c * w2c - w2s * w2s, w4s = 2 * w2c * w2s;  // W_n^kk (= -1 at kk = i)
        const int a1 = kk == i ? 0 : kk, a2 = (kk == 0 || kk == i) ? 0 : i - kk;
        const T c2 = (kk == 0) ? (T)1 : w4c, s2 = (kk == 0) ? (T)0 : -w4s;
        const T2 ze1 = Ze[a1], ze2 = Ze[a2];
        T o1r, o1i, o2r, o2i;
        xs.ld(a1, o1r, o1i);
        xs.ld(a2, o2r, o2i);
        const T z1r = ze1.x + (o1r * w4c - o1i * w4s), z1i = ze1.y + (o1r * w4s + o1i * w4c);
        const T z2r = ze2.x + (o2r * c2 - o2i * s2), z2i = ze2.y + (o2r * s2 + o2i * c2);
        T2 f1, f2;
        analysis_unpack_pair<T>(z1r, z1i, z2r, z2i, pc, ps, R.shifted, h, f1, f2);
        dst[kk] = f1;
        if (n - kk <= mcut && kk != i) dst[n - kk] = f2;
    }
    // aliased orders m > n (lmax beyond the ring's Nyquist frequency): one at a time
    for (int m = n + 1 + tid; m <= mcut; m += NT) {
        const int k = m < N ? m : m % N;
        const bool cj = k > n;
        const int kk = cj ? N - k : k;
        T pc, ps;  // omega^kk
        rt.template get<-1>(kk, pc, ps);
        const T w2c = pc * pc - ps * ps, w2s = 2 * pc * ps;      // W_N^kk
        const T w4c = w2c * w2c - w2s * w2s, w4s = 2 * w2c * w2s;  // W_n^kk
        const int q1 = kk == n ? 0 : kk, q2 = kk == 0 ? 0 : n - kk;
        const int a1 = q1 >= i ? q1 - i : q1, a2 = q2 >= i ? q2 - i : q2;
        // W_n^(n - kk) = conj(W_n^kk); W_n^0 = 1
        const T c1 = (kk == n) ? (T)1 : w4c, s1 = (kk == n) ? (T)0 : w4s;
        const T c2 = (kk == 0) ? (T)1 : w4c, s2 = (kk == 0) ? (T)0 : -w4s;
        const T2 ze1 = Ze[a1], ze2 = Ze[a2];
        T o1r, o1i, o2r, o2i;
        xs.ld(a1, o1r, o1i);
        xs.ld(a2, o2r, o2i);
        const T z1r = ze1.x + (o1r * c1 - o1i * s1), z1i = ze1.y + (o1r * s1 + o1i * c1);
        const T z2r = ze2.x + (o2r * c2 - o2i * s2), z2i = ze2.y + (o2r * s2 + o2i * c2);
        const T er = (T)0.5 * (z1r + z2r), ei = (T)0.5 * (z1i - z2i);
        const T dr = (T)0.5 * (z1r - z2r), di = (T)0.5 * (z1i + z2i);
        T xr = er + (w2c * di + w2s * dr);
        T xi = ei + (w2s * di - w2c * dr);
        if (cj) xi = -xi;
        if (R.shifted) {
            T tc = pc, ts = ps;
            if (k != m || cj) rt.template get<-1>(m % Q, tc, ts);  // aliased: twist != omega^kk
            const T tr = xr * tc - xi * ts, ti = xr * ts + xi * tc;
            xr = tr;
            xi = ti;
        }
        T2 o;
        o.x = wt * xr;
        o.y = wt * xi;
        dst[m] = o;
    }
}

template <typename T, int LOGM>
__global__ void __launch_bounds__(FftPlan<LOGM>::NT, MinBlocks<T, LOGM>::blue) ring_blue_synthesis_kernel(DevPlan P, const RingInfo* __restrict__ info,
                                                                                T* __restrict__ map,
                                                                                const double* __restrict__ w, int use_w,
                                                                                FftTables tabs) {
    if (!ws_ok(P)) return;
    using F = BlockFFT<T, LOGM>;
    using T2 = typename V2<T>::type;
    using SM = BlueSmem<T, LOGM>;
    constexpr int M = F::N, E = F::E, NT = F::NT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Xchg<T> xs(smem_raw, M);
    T2* De = reinterpret_cast<T2*>(smem_raw + SM::off_z);
    T2* rq = reinterpret_cast<T2*>(smem_raw + SM::off_rq);
    T2* rm = reinterpret_cast<T2*>(smem_raw + SM::off_rm);
    const int tid = threadIdx.x;
    const int ch = blockIdx.y;
    const RingInfo R = begin_item<T, false>(P, info, map, tabs.pf);
    prefetch_filter<T>(info, tabs, M);
    const int N = R.N, i = N >> 2, n = N >> 1, Q = 2 * N;
    const T2* filt = reinterpret_cast<const T2*>(tabs.filt) + __ldg(tabs.filt_offset + i);
    fill_roots_any<T>(rq, Q, tid, NT);
    fill_roots_pow2<T>(rm, M, reinterpret_cast<const T2*>(tabs.tw), tabs.twlen, tid, NT);
    const T wt = (T)ring_weight(P, R, w, use_w);
    const float inv_twoi = 1.0f / (float)(2 * i);
    __syncthreads();
    const Roots<T> rt(rq), rtM(rm);
    T2* cs = reinterpret_cast<T2*>(smem_raw + SM::off_cs) + tid;  // [e * NT]: private to this thread
    if constexpr (SM::KEEP_CHIRP) {
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int u = F::index0(tid, e);
            T2 v;
            v.x = 1;
            v.y = 0;
            if (u < i) rt.template get<-1>(chirp_index(u, 2 * i, inv_twoi), v.x, v.y);
            cs[e * NT] = v;
        }
    }
    const T2* G = reinterpret_cast<const T2*>(P.spectra) + ((size_t)ch * P.nrings + R.r) * P.mstride;
    T re[E], im[E];
#pragma unroll 1
    for (int sub = 0; sub < 2; ++sub) {
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int u = F::index0(tid, e);
            re[e] = 0;
            im[e] = 0;
            if (u < i) {
                T yr, yi;
                synth_packed_input<T, false>(G, 2 * u + sub, N, R.mcut, R.shifted, rt, yr, yi);
                T c, s;
                if constexpr (SM::KEEP_CHIRP) {
                    const T2 v = cs[e * NT];
                    c = v.x;
                    s = v.y;
                } else {
                    rt.template get<-1>(chirp_index(u, 2 * i, inv_twoi), c, s);
                }
                re[e] = yr * c - yi * s;
                im[e] = yr * s + yi * c;
            }
        }
        chirp_convolve<T, LOGM>(re, im, xs, rtM, filt, tid);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int u = F::index0(tid, e);
            if (u < i) {
                T c, s;
                if constexpr (SM::KEEP_CHIRP) {
                    const T2 v = cs[e * NT];
                    c = v.x;
                    s = v.y;
                } else {
                    rt.template get<-1>(chirp_index(u, 2 * i, inv_twoi), c, s);
                }
                const T vr = re[e] * c - im[e] * s, vi = re[e] * s + im[e] * c;
                if (sub == 0) {
                    T2 v;
                    v.x = vr;
                    v.y = vi;
                    De[u] = v;
                } else {
                    xs.st(u, vr, vi);
                }
            }
        }
    }
    __syncthreads();
    // D[t] = De[t mod i] + W_n^t Do[t mod i];  x[2t] = Re D[t], x[2t+1] = -Im D[t]
    T2* dst = reinterpret_cast<T2*>(map + (size_t)ch * P.npix + R.start);
#pragma unroll 4
    for (int t = tid; t < n; t += NT) {
        const int ti = t >= i ? t - i : t;
        T c, s;
        rt.template get<-1>(4 * t, c, s);
        const T2 de = De[ti];
        T orr, oi;
        xs.ld(ti, orr, oi);
        T2 o;
        o.x = wt * (de.x + (orr * c - oi * s));
        o.y = -wt * (de.y + (orr * s + oi * c));
        dst[t] = o;
    }
}

// Filter spectrum of cap-ring size i:  b[j] = exp(+i pi j^2 / i) for |j| < i (wrapped into length M), else 0;
// filt = FFT_M(b) / M in the register order of BlockFFT<T, LOGM> ([e][tid]).  Computed in fp64, stored as T.
template <typename T, int LOGM>
__global__ void __launch_bounds__(FftPlan<LOGM>::NT) blue_filter_kernel(const int* __restrict__ ivals,
                                                                        const long long* __restrict__ offsets,
                                                                        typename V2<T>::type* __restrict__ out,
                                                                        const double2* __restrict__ tw64, int twlen) {
    using F = BlockFFT<double, LOGM>;
    constexpr int M = F::N, E = F::E, NT = F::NT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Xchg<double> xs(smem_raw, M);
    double2* rm = reinterpret_cast<double2*>(smem_raw + Xchg<double>::bytes(M));
    const int tid = threadIdx.x;
    const int i = ivals[blockIdx.x];
    fill_roots_pow2<double>(rm, M, tw64, twlen, tid, NT);
    __syncthreads();
    const Roots<double> rtM(rm);
    double re[E], im[E];
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int idx = F::index0(tid, e);
        int j = -1;
        if (idx < i) j = idx;
        else if (M - idx < i) j = M - idx;
        re[e] = 0;
        im[e] = 0;
        if (j >= 0) {
            double c, s;
            cispi_ratio((long long)((j * j) % (2 * i)), i, 1.0, c, s);
            re[e] = c;
            im[e] = s;
        }
    }
    F::forward(re, im, xs, rtM, tid);
    typename V2<T>::type* dst = out + offsets[i];
#pragma unroll
    for (int e = 0; e < E; ++e) {
        typename V2<T>::type v;
        v.x = (T)(re[e] * (1.0 / M));
        v.y = (T)(im[e] * (1.0 / M));
        dst[e * NT + tid] = v;
    }
}

template <typename T>
__global__ void twiddle_table_kernel(typename V2<T>::type* tw, int twlen) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < twlen) {
        double s, c;
        sincospi(-2.0 * (double)k / (double)twlen, &s, &c);
        tw[k].x = (T)c;
        tw[k].y = (T)s;
    }
}

// ------------------------------------------------------------------ planning (host only: a pure function of the call parameters)
static int blue_logm(int i) {  // M = 2^LOGM >= 2 i - 1, at least 2^MIN_LOG
    int l = ilog2_ceil(2LL * i - 1);
    return l < MIN_LOG ? MIN_LOG : l;
}

template <typename T, int LOG> static size_t fft_smem_bytes(bool blue) {
    if (blue) return BlueSmem<T, LOG>::total;
    return Xchg<T>::bytes(1 << LOG) + sizeof(T) * 2 * (size_t)roots_len(4 << LOG);
}
constexpr int HALVES_LOG = 13;  // packed-FFT size class whose fp64 rings are processed in halves
// exchange buffer(s) of H = 2^LOGH points + root table of order Q = 8 H
template <typename T, int LOGH> static size_t half_smem_bytes(int teams) {
    return teams * Xchg<T>::bytes(1 << LOGH) + sizeof(T) * 2 * (size_t)roots_len(8 << LOGH);
}
template <int LOG> static size_t filter_smem_bytes() {
    return Xchg<double>::bytes(1 << LOG) + sizeof(double2) * (size_t)roots_len(1 << LOG);
}

bool fft_supported(int max_ring_pixels, cuhpx_dtype_t dt) {
    (void)dt;
    return max_ring_pixels <= 16384;  // belt: n = N / 2 <= 2^13; caps: M <= 2^13 (fp64 needs 209 KB of the SM's 227 KB)
}

// Host part of the FFT-stage plan: ring classes and the layout of the tables inside the workspace (offsets relative to
// the FFT region, HostPlan::off_fft):
//   [work items: direct | pow2[7..13] | blue[7..13]] [blue_i[7..13]] [filt_offset: nside x i64]
//   [twiddle T2[twlen]] [twiddle double2[twlen] (set-up only, kept)] [filters]
struct FftHost {
    std::vector<RingInfo> direct;
    std::vector<RingInfo> pow2[MAX_LOG + 1];
    std::vector<RingInfo> blue[MAX_LOG + 1];
    std::vector<int> blue_i[MAX_LOG + 1];  // distinct i per LOGM
    std::vector<long long> filt_off;       // [nside] offset (complex units) of the filter of cap ring i, -1 if none
    size_t off_direct, off_pow2[MAX_LOG + 1], off_blue[MAX_LOG + 1], off_blue_i[MAX_LOG + 1];
    size_t off_filt_offset, off_tw, off_tw64, off_filt, total;
    long long filt_total;
    int twlen;
    int max_mcut_direct;
    int pow2_max_mcut;  // largest order wanted on a belt ring
    int side_from;  // Bluestein classes with LOG <= side_from go to the side stream (with the direct kernel)
};
void free_fft_host(FftHost* f) { delete f; }

size_t fft_plan_host(HostPlan& hp) {
    const DevPlan& d = hp.d;
    FftHost* F = new FftHost;
    free_fft_host(hp.fft);
    hp.fft = F;
    for (int r = 0; r < d.nrings; ++r) {
        const int j = std::min(r, d.nrings - 1 - r);
        RingInfo R;
        R.N = hp.h_ringN[j];
        R.start = (r > j) ? d.npix - R.N - hp.h_start[j] : hp.h_start[j];
        R.mcut = hp.h_mcut[j];
        R.shifted = hp.h_shifted[j];
        R.r = r;
        R.pad0 = R.pad1 = 0;
        const int N = R.N;
        // the longest rings when their length is 2^k: HEALPix belt rings (N = 4 nside), every ring of an iso-latitude grid
        if (N == hp.max_ring && is_pow2(N) && ilog2_ceil(N) - 1 >= MIN_LOG) F->pow2[ilog2_ceil(N) - 1].push_back(R);
        else if (N <= DIRECT_MAX_N) F->direct.push_back(R);
        else {  // cap rings, chirp-z for every i (the few i = 2^k among them are not worth launches of their own)
            const int i = N / 4, lm = blue_logm(i);
            F->blue[lm].push_back(R);
            if (r == j) F->blue_i[lm].push_back(i);
        }
    }
    // longest rings first inside a class: the tail of a launch is then made of its cheapest items
    for (int l = MIN_LOG; l <= MAX_LOG; ++l)
        std::stable_sort(F->blue[l].begin(), F->blue[l].end(), [](const RingInfo& a, const RingInfo& b) { return a.N > b.N; });

    const size_t csize = hp.dtype == CUHPX_F64 ? 16 : 8;
    size_t o = 0;
    auto take = [&](size_t bytes) {
        size_t r = o;
        o = (o + bytes + 255) / 256 * 256;
        return r;
    };
    F->off_direct = take(sizeof(RingInfo) * F->direct.size());
    for (int l = 0; l <= MAX_LOG; ++l) F->off_pow2[l] = F->off_blue[l] = F->off_blue_i[l] = 0;
    for (int l = MIN_LOG; l <= MAX_LOG; ++l) {
        F->off_pow2[l] = take(sizeof(RingInfo) * F->pow2[l].size());
        F->off_blue[l] = take(sizeof(RingInfo) * F->blue[l].size());
        F->off_blue_i[l] = take(sizeof(int) * F->blue_i[l].size());
    }
    const int nfilt = hp.max_ring / 4 > 0 ? hp.max_ring / 4 : 1;  // cap rings have N = 4 i, i < nfilt
    F->off_filt_offset = take(sizeof(long long) * nfilt);
    F->twlen = 2 * hp.max_ring < 2048 ? 2048 : 2 * hp.max_ring;
    F->off_tw = take(csize * F->twlen);
    F->off_tw64 = take(16 * (size_t)F->twlen);
    F->filt_off.assign(nfilt, -1);
    long long fo = 0;
    for (int l = MIN_LOG; l <= MAX_LOG; ++l)
        for (int i : F->blue_i[l]) {
            F->filt_off[i] = fo;
            fo += 1LL << l;
        }
    F->filt_total = fo;
    F->off_filt = take(csize * (size_t)fo);
    F->total = o;
    F->max_mcut_direct = 0;
    F->pow2_max_mcut = 0;
    for (int l = MIN_LOG; l <= MAX_LOG; ++l)
        for (const RingInfo& R : F->pow2[l]) F->pow2_max_mcut = std::max(F->pow2_max_mcut, R.mcut);
    for (const RingInfo& R : F->direct) F->max_mcut_direct = std::max(F->max_mcut_direct, R.mcut);
    int lmax_blue = -1;
    for (int l = MIN_LOG; l <= MAX_LOG; ++l)
        if (!F->blue[l].empty()) lmax_blue = l;
    F->side_from = lmax_blue - 2;
    return F->total;
}

// ------------------------------------------------------------------ per-device lazily created launch resources
// Kernel attributes (dynamic shared memory), L2-prefetch distances (CTAs resident on the whole GPU) and the side
// stream on which the short-ring classes run beside the long-ring kernels (fork / join with events, so their launch
// latencies and partial waves hide under the kernels that carry the bytes).  None of it belongs to a workspace.
struct DevRes {
    bool ready = false;
    cudaError_t err = cudaSuccess;
    // [dtype f32 0 / f64 1][analysis 0 / synthesis 1][pow2 0 / blue 1][LOG]
    int pf[2][2][2][MAX_LOG + 1];
    cudaStream_t side = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    std::mutex mu;  // the (record, wait) pairs on the shared events must not interleave between host threads
};
static DevRes g_dev[64];
static std::mutex g_dev_mu;

template <typename T, int LOG> static cudaError_t set_smem_attrs(DevRes& D, int sms) {
    cudaError_t e;
    constexpr int TI = sizeof(T) == 8 ? 1 : 0;
    const size_t sp = fft_smem_bytes<T, LOG>(false), sb = fft_smem_bytes<T, LOG>(true);
    if ((e = cudaFuncSetAttribute(ring_pow2_analysis_kernel<T, LOG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sp))) return e;
    if ((e = cudaFuncSetAttribute(ring_pow2_synthesis_kernel<T, LOG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sp))) return e;
    if ((e = cudaFuncSetAttribute(ring_blue_analysis_kernel<T, LOG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb))) return e;
    if ((e = cudaFuncSetAttribute(ring_blue_synthesis_kernel<T, LOG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb))) return e;
    if ((e = cudaFuncSetAttribute(blue_filter_kernel<T, LOG>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)filter_smem_bytes<LOG>()))) return e;
    int occ = 0;
    constexpr int NT = FftPlan<LOG>::NT;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, ring_pow2_analysis_kernel<T, LOG>, NT, sp))) return e;
    D.pf[TI][0][0][LOG] = occ * sms;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, ring_pow2_synthesis_kernel<T, LOG>, NT, sp))) return e;
    D.pf[TI][1][0][LOG] = occ * sms;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, ring_blue_analysis_kernel<T, LOG>, NT, sb))) return e;
    D.pf[TI][0][1][LOG] = occ * sms;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, ring_blue_synthesis_kernel<T, LOG>, NT, sb))) return e;
    D.pf[TI][1][1][LOG] = occ * sms;
    return cudaSuccess;
}

template <typename T> static cudaError_t set_all_attrs(DevRes& D, int sms) {
    cudaError_t e;
#define CUHPX_ATTR(LOG) if ((e = set_smem_attrs<T, LOG>(D, sms)) != cudaSuccess) return e;
    CUHPX_ATTR(7) CUHPX_ATTR(8) CUHPX_ATTR(9) CUHPX_ATTR(10) CUHPX_ATTR(11) CUHPX_ATTR(12) CUHPX_ATTR(13)
#undef CUHPX_ATTR
    if constexpr (sizeof(T) == 8) {
        if ((e = cudaFuncSetAttribute(ring_pow2_half_analysis_kernel<T, HALVES_LOG - 1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (int)half_smem_bytes<T, HALVES_LOG - 1>(1)))) return e;
        if ((e = cudaFuncSetAttribute(ring_pow2_teams_synthesis_kernel<T, HALVES_LOG - 1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (int)half_smem_bytes<T, HALVES_LOG - 1>(2)))) return e;
    }
    // direct synthesis kernel: [twiddles N][G: mcut + 1]; the largest the SM can hold (launches check their own need)
    return cudaFuncSetAttribute(ring_direct_synthesis_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
}

static DevRes* dev_res(cudaError_t* err) {
    int dev = 0;
    if ((*err = cudaGetDevice(&dev)) != cudaSuccess) return nullptr;
    if (dev < 0 || dev >= 64) {
        *err = cudaErrorInvalidDevice;
        return nullptr;
    }
    DevRes& D = g_dev[dev];
    std::lock_guard<std::mutex> lk(g_dev_mu);
    if (!D.ready) {
        int sms = 0;
        cudaError_t e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        memset(D.pf, 0, sizeof(D.pf));
        if (e == cudaSuccess) e = set_all_attrs<float>(D, sms);
        if (e == cudaSuccess) e = set_all_attrs<double>(D, sms);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&D.side, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&D.ev_fork, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&D.ev_join, cudaEventDisableTiming);
        D.err = e;
        D.ready = true;
    }
    *err = D.err;
    return D.err == cudaSuccess ? &D : nullptr;
}

// ------------------------------------------------------------------ table building (cuhpx_workspace_init)
template <typename T, int LOG>
static cudaError_t build_filters(const FftHost& F, char* base, cudaStream_t st) {
    if (F.blue_i[LOG].empty()) return cudaSuccess;
    using T2 = typename V2<T>::type;
    blue_filter_kernel<T, LOG><<<(unsigned)F.blue_i[LOG].size(), FftPlan<LOG>::NT, filter_smem_bytes<LOG>(), st>>>(
        (const int*)(base + F.off_blue_i[LOG]), (const long long*)(base + F.off_filt_offset), (T2*)(base + F.off_filt),
        (const double2*)(base + F.off_tw64), F.twlen);
    return cudaGetLastError();
}

template <typename T> static cudaError_t build_tables_t(const FftHost& F, char* base, cudaStream_t st) {
    using T2 = typename V2<T>::type;
    cudaError_t e;
    twiddle_table_kernel<T><<<(F.twlen + 255) / 256, 256, 0, st>>>((T2*)(base + F.off_tw), F.twlen);
    twiddle_table_kernel<double><<<(F.twlen + 255) / 256, 256, 0, st>>>((double2*)(base + F.off_tw64), F.twlen);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
#define CUHPX_FILT(LOG) if ((e = build_filters<T, LOG>(F, base, st)) != cudaSuccess) return e;
    CUHPX_FILT(7) CUHPX_FILT(8) CUHPX_FILT(9) CUHPX_FILT(10) CUHPX_FILT(11) CUHPX_FILT(12) CUHPX_FILT(13)
#undef CUHPX_FILT
    return cudaSuccess;
}

cudaError_t fft_build_tables(const HostPlan& hp, char* base, cudaStream_t st) {
    if (!hp.fft) return cudaErrorInvalidValue;
    const FftHost& F = *hp.fft;
    cudaError_t e = cudaSuccess;
    if (!dev_res(&e)) return e;  // kernel attributes of this device are in place before the first (possibly captured) call
    const size_t csz = hp.dtype == CUHPX_F64 ? 16 : 8;
    if ((DIRECT_MAX_N + F.max_mcut_direct + 1) * csz > 200 * 1024) return cudaErrorInvalidConfiguration;
    auto up = [&](size_t off, const void* src, size_t bytes) {
        if (e == cudaSuccess && bytes) e = cudaMemcpyAsync(base + off, src, bytes, cudaMemcpyHostToDevice, st);
    };
    up(F.off_direct, F.direct.data(), sizeof(RingInfo) * F.direct.size());
    for (int l = MIN_LOG; l <= MAX_LOG; ++l) {
        up(F.off_pow2[l], F.pow2[l].data(), sizeof(RingInfo) * F.pow2[l].size());
        up(F.off_blue[l], F.blue[l].data(), sizeof(RingInfo) * F.blue[l].size());
        up(F.off_blue_i[l], F.blue_i[l].data(), sizeof(int) * F.blue_i[l].size());
    }
    up(F.off_filt_offset, F.filt_off.data(), sizeof(long long) * F.filt_off.size());
    if (e != cudaSuccess) return e;
    return hp.dtype == CUHPX_F64 ? build_tables_t<double>(F, base, st) : build_tables_t<float>(F, base, st);
}

void fft_stage_stats(const HostPlan& hp, int* launches, double* table_bytes) {
    *launches = 0;
    *table_bytes = 0;
    if (!hp.fft) return;
    const FftHost& F = *hp.fft;
    const double csz = hp.dtype == CUHPX_F64 ? 16 : 8;
    if (!F.direct.empty()) ++*launches;
    for (int l = MIN_LOG; l <= MAX_LOG; ++l) {
        if (!F.pow2[l].empty()) ++*launches;
        if (!F.blue[l].empty()) {
            ++*launches;
            *table_bytes += 0.5 * F.blue[l].size() * (double)(1 << l) * csz;  // one filter per ring size i, shared N/S
        }
    }
    *table_bytes += F.twlen * csz;
}

// ------------------------------------------------------------------ launchers
struct FftCall {  // what one stage call resolves from (plan, workspace, device)
    const FftHost* F;
    const char* base;  // FFT region of the workspace
    const DevRes* D;
    FftTables tabs;
    int ti;  // 0 fp32, 1 fp64
};

// Bluestein classes LOG <= side_from and the direct kernel go to the side stream
template <typename T, bool ANALYSIS, int LOG>
static void launch_class(const DevPlan& P, const FftCall& C, T* map, const double* w, int use_w, cudaStream_t main_st,
                         cudaStream_t side_st) {
    const FftHost& F = *C.F;
    FftTables tabs = C.tabs;
    constexpr int A = ANALYSIS ? 0 : 1;
    if (!F.pow2[LOG].empty()) {
        tabs.pf = C.D->pf[C.ti][A][0][LOG];
        const RingInfo* items = (const RingInfo*)(C.base + F.off_pow2[LOG]);
        const unsigned ni = (unsigned)F.pow2[LOG].size();
        const dim3 grid(ni, P.batch);
        bool done = false;
        if constexpr (LOG == HALVES_LOG && sizeof(T) == 8) {
            // fp64 rings of 2^14 pixels: half-ring work items / two teams per CTA (unless orders beyond the ring's
            // Nyquist frequency are wanted: those need both halves of the spectrum in one place)
            if (F.pow2_max_mcut <= (2 << LOG) / 2) {
                if (ANALYSIS)
                    ring_pow2_half_analysis_kernel<T, LOG - 1><<<dim3(2 * ni, P.batch), FftPlan<LOG - 1>::NT, half_smem_bytes<T, LOG - 1>(1), main_st>>>(
                        P, items, map, w, use_w, tabs);
                else
                    ring_pow2_teams_synthesis_kernel<T, LOG - 1><<<grid, 2 * FftPlan<LOG - 1>::NT, half_smem_bytes<T, LOG - 1>(2), main_st>>>(
                        P, items, map, w, use_w, tabs);
                done = true;
            }
        }
        if (done) {
        } else if (ANALYSIS)
            ring_pow2_analysis_kernel<T, LOG><<<grid, FftPlan<LOG>::NT, fft_smem_bytes<T, LOG>(false), main_st>>>(P, items, map, w, use_w, tabs);
        else
            ring_pow2_synthesis_kernel<T, LOG><<<grid, FftPlan<LOG>::NT, fft_smem_bytes<T, LOG>(false), main_st>>>(P, items, map, w, use_w, tabs);
    }
    if (!F.blue[LOG].empty()) {
        tabs.pf = C.D->pf[C.ti][A][1][LOG];
        cudaStream_t st = LOG <= F.side_from ? side_st : main_st;
        const RingInfo* items = (const RingInfo*)(C.base + F.off_blue[LOG]);
        const dim3 grid((unsigned)F.blue[LOG].size(), P.batch);
        if (ANALYSIS)
            ring_blue_analysis_kernel<T, LOG><<<grid, FftPlan<LOG>::NT, fft_smem_bytes<T, LOG>(true), st>>>(P, items, map, w, use_w, tabs);
        else
            ring_blue_synthesis_kernel<T, LOG><<<grid, FftPlan<LOG>::NT, fft_smem_bytes<T, LOG>(true), st>>>(P, items, map, w, use_w, tabs);
    }
}

template <typename T, bool ANALYSIS>
static cudaError_t run_fft_stage(const HostPlan& hp, const DevPlan& P, T* map, const double* d_w, int use_w, cudaStream_t st) {
    if (!hp.fft) return cudaErrorInvalidValue;
    cudaError_t e = cudaSuccess;
    DevRes* D = dev_res(&e);
    if (!D) return e;
    const FftHost& F = *hp.fft;
    FftCall C;
    C.F = &F;
    C.base = reinterpret_cast<const char*>(P.hdr) + hp.off_fft;
    C.D = D;
    C.ti = sizeof(T) == 8 ? 1 : 0;
    C.tabs.tw = C.base + F.off_tw;
    C.tabs.twlen = F.twlen;
    C.tabs.filt = C.base + F.off_filt;
    C.tabs.filt_offset = (const long long*)(C.base + F.off_filt_offset);
    C.tabs.pf = 0;
    bool side_work = !F.direct.empty(), main_work = false;
    for (int l = MIN_LOG; l <= MAX_LOG; ++l) {
        if (!F.blue[l].empty() && l <= F.side_from) side_work = true;
        if (!F.pow2[l].empty() || (!F.blue[l].empty() && l > F.side_from)) main_work = true;
    }
    const bool fork = side_work && main_work;
    cudaStream_t side = fork ? D->side : st;
    std::unique_lock<std::mutex> lk(D->mu, std::defer_lock);
    if (fork) {
        lk.lock();
        if ((e = cudaEventRecord(D->ev_fork, st)) != cudaSuccess) return e;
        if ((e = cudaStreamWaitEvent(side, D->ev_fork, 0)) != cudaSuccess) return e;
    }
    // largest rings first: they dominate the run time
    launch_class<T, ANALYSIS, 13>(P, C, map, d_w, use_w, st, side);
    launch_class<T, ANALYSIS, 12>(P, C, map, d_w, use_w, st, side);
    launch_class<T, ANALYSIS, 11>(P, C, map, d_w, use_w, st, side);
    launch_class<T, ANALYSIS, 10>(P, C, map, d_w, use_w, st, side);
    launch_class<T, ANALYSIS, 9>(P, C, map, d_w, use_w, st, side);
    launch_class<T, ANALYSIS, 8>(P, C, map, d_w, use_w, st, side);
    launch_class<T, ANALYSIS, 7>(P, C, map, d_w, use_w, st, side);
    if (!F.direct.empty()) {
        constexpr int CB = 8;
        const RingInfo* items = (const RingInfo*)(C.base + F.off_direct);
        const unsigned nd = (unsigned)F.direct.size();
        const size_t cb_ana = (size_t)DIRECT_MAX_N * (2 + CB) * sizeof(T);
        const size_t cb_syn = ((size_t)DIRECT_MAX_N + (size_t)(F.max_mcut_direct + 1) * CB) * 2 * sizeof(T);
        if (P.batch >= 4 && cb_syn <= 48 * 1024) {  // channel-blocked direct sums
            const dim3 grid(nd, (P.batch + CB - 1) / CB);
            if (ANALYSIS) ring_direct_analysis_cb_kernel<T, CB><<<grid, DIRECT_CB_THREADS, cb_ana, side>>>(P, items, map, d_w, use_w);
            else ring_direct_synthesis_cb_kernel<T, CB><<<grid, DIRECT_CB_THREADS, cb_syn, side>>>(P, items, map, d_w, use_w);
        } else if (ANALYSIS)
            ring_direct_analysis_kernel<T><<<dim3(nd, P.batch), FFT_THREADS, (size_t)DIRECT_MAX_N * 3 * sizeof(T), side>>>(
                P, items, map, d_w, use_w);
        else
            ring_direct_synthesis_kernel<T><<<dim3(nd, P.batch), FFT_THREADS,
                                              ((size_t)DIRECT_MAX_N + F.max_mcut_direct + 1) * 2 * sizeof(T), side>>>(P, items, map, d_w, use_w);
    }
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if (fork) {
        if ((e = cudaEventRecord(D->ev_join, side)) != cudaSuccess) return e;
        if ((e = cudaStreamWaitEvent(st, D->ev_join, 0)) != cudaSuccess) return e;
    }
    return cudaSuccess;
}

cudaError_t launch_fft_analysis(const HostPlan& hp, const DevPlan& P, const void* d_map, const double* d_w, int use_w,
                                cudaStream_t st) {
    // analysis kernels only read the map; one launcher template serves both directions
    return hp.dtype == CUHPX_F64 ? run_fft_stage<double, true>(hp, P, (double*)const_cast<void*>(d_map), d_w, use_w, st)
                                 : run_fft_stage<float, true>(hp, P, (float*)const_cast<void*>(d_map), d_w, use_w, st);
}

cudaError_t launch_fft_synthesis(const HostPlan& hp, const DevPlan& P, void* d_map, const double* d_w, int use_w,
                                 cudaStream_t st) {
    return hp.dtype == CUHPX_F64 ? run_fft_stage<double, false>(hp, P, (double*)d_map, d_w, use_w, st)
                                 : run_fft_stage<float, false>(hp, P, (float*)d_map, d_w, use_w, st);
}

}  // namespace cuhpx

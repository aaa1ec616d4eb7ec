// Legendre stage of the HEALPix SHT:
//   analysis : a_lm = sum_j lambda_lm(theta_j) [F_m(N_j) + (-1)^(l+m) F_m(S_j)]          (Eq. 14, Eq. 26)
//   synthesis: G_m(N_j) = E + O, G_m(S_j) = E - O,  E/O = sum_{l, (l+m) even/odd} a_lm lambda_lm(theta_j)  (Eq. 24)
// lambda_lm is generated on the fly by the three-term recurrence of Eq. 16 from exponent-scaled
// seeds lambda_mm (Eq. 15); nothing is precomputed per (l, m, ring) -- the paper's stored Legendre
// tensor and its out-of-core streaming do not exist here.
//
// Thread mapping: one block = one m, one chunk of ring pairs, one group of BT channels.  Each thread owns R
// ring pairs (lanes = adjacent rings) and walks l = m .. lmax carrying (lambda_{l}, lambda_{l-1}) in fp64
// registers.  cos(theta) enters as x p = p - y p with y = 1 - cos(theta) (R3).
#include <cuda_runtime.h>
#include <math.h>
#include <stdlib.h>

#include "cuhpx_internal.h"
#include "legendre_common.cuh"

namespace cuhpx {

constexpr int CT = 64;  // recurrence-coefficient tile (l values per __syncthreads)

// ------------------------------------------------------------------ recurrence coefficients (built once per plan)
// Eq. 16 reads lambda_l = A_l x lambda_{l-1} + B_l lambda_{l-2}, A_l = sqrt((4l^2-1)/(l^2-m^2)),
// B_l = -sqrt((2l+1)/(2l-3) ((l-1)^2-m^2)/(l^2-m^2)).  The kernels iterate the diagonally rescaled sequence
// mu_l = lambda_l / s_l with s_m = s_{m+1} = 1, s_l = |B_l| s_{l-2}, for which
//        mu_l = alpha_l x mu_{l-1} - mu_{l-2},   alpha_l = A_l s_{l-1} / s_l,
// i.e. two FMAs per degree instead of mul + mul + FMA; s_l is applied once per coefficient (to a_lm before the
// synthesis sum, to the reduced sum after the analysis).  alpha must be good to an ulp (near the poles the
// recurrence amplifies coefficient errors by ~1/theta^2, R3), so the table is built in double-double.
struct dd {
    double hi, lo;
};
__device__ __forceinline__ dd dd_from(double a) { return dd{a, 0.0}; }
__device__ __forceinline__ dd dd_two_prod(double a, double b) {
    const double p = a * b;
    return dd{p, fma(a, b, -p)};
}
__device__ __forceinline__ dd dd_norm(double hi, double lo) {
    const double s = hi + lo;
    return dd{s, lo - (s - hi)};
}
__device__ __forceinline__ dd dd_mul(dd a, dd b) {
    dd p = dd_two_prod(a.hi, b.hi);
    p.lo += a.hi * b.lo + a.lo * b.hi;
    return dd_norm(p.hi, p.lo);
}
__device__ __forceinline__ dd dd_div(dd a, dd b) {
    const double q1 = a.hi / b.hi;
    // r = a - q1 * b
    dd p = dd_mul(dd_from(q1), b);
    const double r = (a.hi - p.hi) + (a.lo - p.lo);
    const double q2 = r / b.hi;
    return dd_norm(q1, q2);
}
__device__ __forceinline__ dd dd_sqrt(dd a) {
    if (a.hi <= 0.0) return dd{0.0, 0.0};
    const double x = sqrt(a.hi);
    // one Newton step: x + (a - x^2) / (2x)
    const dd x2 = dd_two_prod(x, x);
    const double r = (a.hi - x2.hi) + (a.lo - x2.lo);
    return dd_norm(x, r / (2.0 * x));
}

// one thread per m; alpha[idx(l,m)], scale[idx(l,m)] for l = m..lmax (alpha[idx(m,m)] = 0: no step produces lambda_mm)
__global__ void legendre_coeff_kernel(int lmax, int mmax, double* __restrict__ alpha, double* __restrict__ scale) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m > mmax) return;
    const long long base = (long long)m * (2LL * lmax + 1 - m) / 2;
    alpha[base + m] = 0.0;
    scale[base + m] = 1.0;
    dd s1 = dd_from(1.0), s2 = dd_from(1.0);  // s_{l-1}, s_{l-2}
    const double dm = (double)m;
    for (int l = m + 1; l <= lmax; ++l) {
        const double dl = (double)l;
        const double l2m2 = (dl - dm) * (dl + dm);  // exact integers below 2^53
        const dd A = dd_sqrt(dd_div(dd_from(4.0 * dl * dl - 1.0), dd_from(l2m2)));
        dd sl = dd_from(1.0);
        if (l >= m + 2) {
            const dd num = dd_two_prod(2.0 * dl + 1.0, (dl - 1.0 - dm) * (dl - 1.0 + dm));
            const dd den = dd_two_prod(2.0 * dl - 3.0, l2m2);
            sl = dd_mul(dd_sqrt(dd_div(num, den)), s2);  // |B_l| s_{l-2}
        }
        const dd al = dd_div(dd_mul(A, s1), sl);
        alpha[base + l] = al.hi + al.lo;
        scale[base + l] = sl.hi + sl.lo;
        s2 = s1;
        s1 = sl;
    }
}

cudaError_t launch_legendre_coeff(int lmax, int mmax, double* alpha, double* scale, cudaStream_t st) {
    legendre_coeff_kernel<<<(mmax + 1 + 63) / 64, 64, 0, st>>>(lmax, mmax, alpha, scale);
    return cudaGetLastError();
}


// sum NV per-thread values across the 32 lanes; afterwards lane L holds, in v[0 .. Q-1], the totals of the
// values with index Q * (L >> SH) + q, Q = max(NV / 32, 1), SH = max(5 - log2 NV, 0).
template <typename T, int NV>
__device__ __forceinline__ void warp_transpose_reduce(T (&v)[NV], int lane) {
    int n = NV;
#pragma unroll
    for (int mask = 16; mask >= 1; mask >>= 1) {
        if (n > 1) {
            const int h = n / 2;
            const bool up = (lane & mask) != 0;
#pragma unroll
            for (int i = 0; i < NV / 2; ++i) {
                if (i < h) {
                    const T send = up ? v[i] : v[i + h];
                    const T keep = up ? v[i + h] : v[i];
                    v[i] = keep + __shfl_xor_sync(0xffffffffu, send, mask);
                }
            }
            n = h;
        } else {
            v[0] += __shfl_xor_sync(0xffffffffu, v[0], mask);
        }
    }
}

// ------------------------------------------------------------------ analysis (row a3)
// Per warp: every LT degrees the NV = LT*BT*2 per-thread partial sums are reduced over the 32 lanes by a
// transposing butterfly and parked in shared memory; every GROUP_L degrees one __syncthreads lets the first
// threads add the warps' values and write a_lm.  The first butterfly level splits (re, im): lanes 16..31 hold
// their F with re and im swapped, so that every lane KEEPS component slot 0 and SENDS slot 1 -- no selects on the
// widest level.  Warps whose rings are all still below the significance threshold skip the accumulation.
constexpr int GROUP_L = 32;  // degrees per cross-warp reduction

// v[2*k + comp], k < NV/2.  After the call lane L holds in v[0 .. Q-1] the 32-lane totals of
// (k = Q * ((L & 15) >> SH) + q, comp = L >> 4), Q = max(NV / 32, 1), SH = max(4 - log2(NV/2), 0).
template <typename T, int NV>
__device__ __forceinline__ void warp_reduce_split(T (&v)[NV], int lane) {
    constexpr int H = NV / 2;
#pragma unroll
    for (int k = 0; k < H; ++k) v[k] = v[2 * k] + __shfl_xor_sync(0xffffffffu, v[2 * k + 1], 16);
    int n = H;
#pragma unroll
    for (int mask = 8; mask >= 1; mask >>= 1) {
        if (n > 1) {
            const int h = n / 2;
            const bool up = (lane & mask) != 0;
#pragma unroll
            for (int i = 0; i < H / 2; ++i) {
                if (i < h) {
                    const T send = up ? v[i] : v[i + h];
                    const T keep = up ? v[i + h] : v[i];
                    v[i] = keep + __shfl_xor_sync(0xffffffffu, send, mask);
                }
            }
            n = h;
        } else {
            v[0] += __shfl_xor_sync(0xffffffffu, v[0], mask);
        }
    }
}

// SEQ: one CTA walks the ring chunks of its order m and accumulates a_lm in place (no partial arrays / combine kernel)
template <typename T, int BT, int R, int LT, int NT, int GL = GROUP_L, bool SEQ = false, int MINB = 384 / NT>
__global__ void __launch_bounds__(NT, MINB) legendre_analysis_kernel(LegArgs a) {
    using T2 = typename Vec2<T>::type;
    constexpr int NW = NT / 32;
    constexpr int NV = LT * BT * 2;
    constexpr int HV = NV / 2;
    constexpr int Q = HV >= 16 ? HV / 16 : 1;
    constexpr int SH = HV >= 16 ? 0 : (HV == 8 ? 1 : HV == 4 ? 2 : HV == 2 ? 3 : 4);
    constexpr int TPG = GL / LT;  // tiles per group
    static_assert(CHECK_EVERY % LT == 0 && CT % GL == 0 && GL % CHECK_EVERY == 0, "tile sizes");
    static_assert(NV >= 4, "reduction tile");
    const DevPlan& P = a.p;
    if (!ws_ok(P)) return;
    const int m = blockIdx.x;
    const int ch0 = blockIdx.z * BT;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    int buf = 0;
    for (int chunk = SEQ ? 0 : (int)blockIdx.y;; ++chunk) {
    const int jbase = P.jmin[m] + chunk * (NT * R);
    if (jbase >= P.npairs) return;

    __shared__ double sA[2][CT];
    __shared__ T red[2][TPG][NW][NV];

    const T2* spectra = reinterpret_cast<const T2*>(P.spectra);
    double cur[R], prev[R], y[R];
    int sc[R];
    // F_N + F_S and F_N - F_S of the ACTIVE rings (zero while inactive); [.][.][0] is the component this lane
    // keeps in the first butterfly level (re for lanes 0-15, im for lanes 16-31), [.][.][1] the one it sends
    T fs[R][BT][2], fa[R][BT][2];
    int nact = 0;
    const double pref_hi = P.pref_hi[m], pref_lo = P.pref_lo[m];
    const bool swap_c = (lane & 16) != 0;

    auto load_F = [&](int r) {
        const int j = jbase + tid + NT * r;
        const int rn = j, rs = P.nrings - 1 - j;
#pragma unroll
        for (int c = 0; c < BT; ++c) {
            const int ch = min(ch0 + c, P.batch - 1);
            const T2 fn = spectra[((size_t)ch * P.nrings + rn) * P.mstride + m];
            T2 fsv;
            fsv.x = 0;
            fsv.y = 0;
            if (rs != rn) fsv = spectra[((size_t)ch * P.nrings + rs) * P.mstride + m];
            const T sr = fn.x + fsv.x, si = fn.y + fsv.y, ar = fn.x - fsv.x, ai = fn.y - fsv.y;
            fs[r][c][0] = swap_c ? si : sr;
            fs[r][c][1] = swap_c ? sr : si;
            fa[r][c][0] = swap_c ? ai : ar;
            fa[r][c][1] = swap_c ? ar : ai;
        }
    };

#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int j = jbase + tid + NT * r;
#pragma unroll
        for (int c = 0; c < BT; ++c) fs[r][c][0] = fs[r][c][1] = fa[r][c][0] = fa[r][c][1] = 0;
        if (j < P.npairs) {
            y[r] = P.y[j];
            lambda_seed<T>(m, pref_hi, pref_lo, P.ls_hi[j], P.ls_lo[j], cur[r], sc[r]);
            prev[r] = 0.0;
            if (sc[r] == 0) {
                load_F(r);
                ++nact;
            }
        } else {  // padding lane: never active, recurrence on zeros
            y[r] = 1.0;
            cur[r] = 0.0;
            prev[r] = 0.0;
            sc[r] = -1;
        }
    }

    const double outscale = (a.adjoint && m > 0) ? 2.0 : 1.0;
    const long long abase = (long long)m * (2LL * P.lmax + 1 - m) / 2;  // index of (l = 0, m) in packed alm
    T* out = reinterpret_cast<T*>(a.out);
    if (a.to_partial) out += (size_t)chunk * P.batch * P.nalm * 2;

    const int nl = P.lmax - m + 1;  // l values of this m
    // late start (tables built by legendre_start_kernel): no ring pair of this chunk is significant before degree
    // m + tstart, so the walk begins there with the recurrence state the skipped steps would have produced
    int tstart = 0;
    if (SEQ && P.st_chunk[0] == NT * R) {
        tstart = P.st_l0[0][(size_t)m * P.st_nchunk[0] + chunk];
        if (tstart > 0) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int j = jbase + tid + NT * r;
                if (j < P.npairs) {
                    const size_t e = (size_t)m * P.npairs + j;
                    cur[r] = P.st_cur[0][e];
                    prev[r] = P.st_prev[0][e];
                    sc[r] = P.st_sc[0][e];
                }
            }
            if (chunk == 0) {  // the first chunk initialises a_lm: zeros where nothing is significant yet
                const int ch = ch0;  // BT == 1 on this path
                if (ch < P.batch)
                    for (int e = tid; e < 2 * tstart; e += NT) out[((size_t)ch * P.nalm + abase + m) * 2 + e] = 0;
            }
        }
    }
    bool warp_active = __any_sync(0xffffffffu, nact > 0);
    // alpha of the steps that produce degrees l = m + t0 + 1 + i; the next tile is fetched into a register while
    // the current one is consumed, so no global-load latency sits between two tiles
    constexpr int APT = (CT + NT - 1) / NT;  // alpha values a thread carries (CTAs may be narrower than the tile)
    double nextA[APT];
#pragma unroll
    for (int q = 0; q < APT; ++q) {
        const int i = tid + q * NT;
        nextA[q] = (i < CT && tstart + 1 + i < nl) ? P.coef_alpha[abase + m + tstart + 1 + i] : 0.0;
    }
    constexpr int NOUT = (TPG * NV + NT - 1) / NT;  // output elements per thread and group (cross-warp sums)
    for (int t0 = tstart; t0 < nl; t0 += CT) {
        const int cb = (t0 / CT) & 1;
#pragma unroll
        for (int q = 0; q < APT; ++q) {
            const int i = tid + q * NT;
            if (i < CT) {
                sA[cb][i] = nextA[q];
                nextA[q] = (t0 + CT + 1 + i < nl) ? P.coef_alpha[abase + m + t0 + CT + 1 + i] : 0.0;
            }
        }
        __syncthreads();
        const int tend = min(CT, nl - t0);
        for (int g0 = 0; g0 < tend; g0 += GL) {
            // s_l of this thread's output element, requested before the group's arithmetic
            double oscl[NOUT];
            T oold[NOUT];  // SEQ: what the earlier ring chunks left in a_lm
#pragma unroll
            for (int q = 0; q < NOUT; ++q) {
                const int e = tid + NT * q;
                const int k = t0 + g0 + (e / NV) * LT + (e % NV) / (BT * 2);
                oscl[q] = (e < TPG * NV && k < nl) ? outscale * P.coef_scale[abase + m + k] : 0.0;
                oold[q] = 0;
                if (SEQ && chunk > 0) {
                    const int v = e % NV, ch = ch0 + (v / 2) % BT;
                    if (e < TPG * NV && k < nl && ch < P.batch) oold[q] = out[((size_t)ch * P.nalm + abase + m + k) * 2 + (v & 1)];
                }
            }
#pragma unroll 1
            for (int ti = 0; ti < TPG; ++ti) {
                const int s0 = g0 + ti * LT;
                if ((s0 % CHECK_EVERY) == 0 && !__all_sync(0xffffffffu, nact == R)) {
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        if (sc[r] < 0 && fabs(cur[r]) > pow2c(ScaleCfg<T>::THR)) {
                            cur[r] *= pow2c(-ScaleCfg<T>::K);
                            prev[r] *= pow2c(-ScaleCfg<T>::K);
                            if (++sc[r] == 0) {
                                load_F(r);
                                ++nact;
                            }
                        }
                    }
                    warp_active = __any_sync(0xffffffffu, nact > 0);
                }
                if (warp_active) {
                    T acc[NV];
#pragma unroll
                    for (int i = 0; i < NV; ++i) acc[i] = 0;
#pragma unroll
                    for (int i = 0; i < LT; ++i) {
                        const double A = sA[cb][s0 + i];
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            const T lam = (T)cur[r];
#pragma unroll
                            for (int c = 0; c < BT; ++c) {
                                // (t0 + s0 + i) = l - m; even -> symmetric combination
                                if (((s0 + i) & 1) == 0) {
                                    acc[(i * BT + c) * 2 + 0] = fma(lam, fs[r][c][0], acc[(i * BT + c) * 2 + 0]);
                                    acc[(i * BT + c) * 2 + 1] = fma(lam, fs[r][c][1], acc[(i * BT + c) * 2 + 1]);
                                } else {
                                    acc[(i * BT + c) * 2 + 0] = fma(lam, fa[r][c][0], acc[(i * BT + c) * 2 + 0]);
                                    acc[(i * BT + c) * 2 + 1] = fma(lam, fa[r][c][1], acc[(i * BT + c) * 2 + 1]);
                                }
                            }
                            const double xl = fma(-y[r], cur[r], cur[r]);
                            const double nx = fma(A, xl, -prev[r]);
                            prev[r] = cur[r];
                            cur[r] = nx;
                        }
                    }
                    warp_reduce_split<T, NV>(acc, lane);
                    if ((lane & ((1 << SH) - 1)) == 0) {
#pragma unroll
                        for (int q = 0; q < Q; ++q)
                            red[buf][ti][warp][2 * (Q * ((lane & 15) >> SH) + q) + (lane >> 4)] = acc[q];
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < LT; ++i) {
                        const double A = sA[cb][s0 + i];
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            const double xl = fma(-y[r], cur[r], cur[r]);
                            const double nx = fma(A, xl, -prev[r]);
                            prev[r] = cur[r];
                            cur[r] = nx;
                        }
                    }
                    for (int v = lane; v < NV; v += 32) red[buf][ti][warp][v] = 0;
                }
            }
            __syncthreads();
#pragma unroll
            for (int q = 0; q < NOUT; ++q) {
                const int e = tid + NT * q;
                if (e >= TPG * NV) break;
                const int ti = e / NV, v = e % NV;
                T sum = 0;
#pragma unroll
                for (int w = 0; w < NW; ++w) sum += red[buf][ti][w][v];
                const int i = v / (BT * 2), c = (v / 2) % BT, ri = v & 1;
                const int k = t0 + g0 + ti * LT + i;  // l - m
                const int ch = ch0 + c;
                if (k < nl && ch < P.batch) {
                    T o = oold[q] + (T)(oscl[q] * (double)sum);  // lambda = s_l mu
                    if (m == 0 && ri == 1) o = 0;  // Im a_l0 is exactly zero
                    out[((size_t)ch * P.nalm + abase + m + k) * 2 + ri] = o;
                }
            }
            buf ^= 1;
        }
    }
    if (!SEQ) return;
    __syncthreads();  // the next chunk reuses the shared tiles
    }  // chunk
}

// ------------------------------------------------------------------ analysis, batched fp32 (row a3 as a contraction)
// With >= 8 channels the Legendre stage really is a dense contraction per m (north_star): C[l][c] = sum_j
// Lambda[l][j] F[j][c], c = (channel, re/im), j = ring pairs.  One CTA = (m, 256 ring pairs, 8 channels): each
// thread walks the recurrence of ONE ring pair in fp64 and parks lambda (fp32, 0 while the ring is insignificant)
// for 32 degrees in shared memory, [parity][ring][16 degrees]; then the CTA multiplies that 32 x 256 tile with the
// resident F tile (F_N + F_S for even l - m, F_N - F_S for odd) as a register-blocked SGEMM: warp = 32 rings of K,
// thread = 4 degrees (one parity) x 4 columns, one LDS.128 of lambda + one of F per 16 FFMA; the 8 warps' partial
// tiles meet in shared memory.  lambda is converted to fp32 once per (l, ring) for all 8 channels.
// packed fp32 FMA of sm_100a (PTX fma.rn.f32x2 -> SASS FFMA2): d = {s * b.x + c.x, s * b.y + c.y} in one issue slot
__device__ __forceinline__ float2 fma2(float s, float2 b, float2 c) {
    float2 d;
    asm("{\n\t.reg .b64 ra, rb, rc, rd;\n\t"
        "mov.b64 ra, {%2, %2};\n\t"
        "mov.b64 rb, {%3, %4};\n\t"
        "mov.b64 rc, {%5, %6};\n\t"
        "fma.rn.f32x2 rd, ra, rb, rc;\n\t"
        "mov.b64 {%0, %1}, rd;\n\t}"
        : "=f"(d.x), "=f"(d.y)
        : "f"(s), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
    return d;
}

constexpr int GK = 256;    // ring pairs per CTA (= threads)
constexpr int GTL = 32;    // degrees per tile
constexpr int GROW = 20;   // floats per lambda row: 16 + 4 padding (conflict-free 16-byte stores at 80-byte pitch)
constexpr int GNCH = 8;    // channels per CTA
constexpr int GNC = 2 * GNCH;

__global__ void __launch_bounds__(GK, 3) legendre_analysis_gemm_kernel(LegArgs a) {
    const DevPlan& P = a.p;
    if (!ws_ok(P)) return;
    const int m = blockIdx.x;
    const int chunk = blockIdx.y;
    const int ch0 = blockIdx.z * GNCH;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int jbase = P.jmin[m] + chunk * GK;
    if (jbase >= P.npairs) return;

    extern __shared__ __align__(16) unsigned char gemm_smem[];
    float* sLam = reinterpret_cast<float*>(gemm_smem);  // [parity][ring][GROW]; reused for the cross-warp sums
    float(*sF)[GK][GNC] = reinterpret_cast<float(*)[GK][GNC]>(sLam + 2 * GK * GROW);  // [0] = F_N + F_S, [1] = F_N - F_S
    double(*sA)[GTL] = reinterpret_cast<double(*)[GTL]>(sLam + 2 * GK * GROW + 2 * GK * GNC);
    double(*sS)[GTL] = sA + 2;  // outscale * s_l of the tile's degrees

    const float2* spectra = reinterpret_cast<const float2*>(P.spectra);
    const int j = jbase + tid;
    const bool valid = j < P.npairs;
    double cur = 0.0, prev = 0.0, y = 1.0;
    int sc = -1;
    {
        float fsum[GNC], fdif[GNC];
#pragma unroll
        for (int c = 0; c < GNC; ++c) fsum[c] = fdif[c] = 0.f;
        if (valid) {
            y = P.y[j];
            lambda_seed<float>(m, P.pref_hi[m], P.pref_lo[m], P.ls_hi[j], P.ls_lo[j], cur, sc);
            const int rn = j, rs = P.nrings - 1 - j;
#pragma unroll
            for (int c = 0; c < GNCH; ++c) {
                if (ch0 + c < P.batch) {
                    const float2 fn = spectra[((size_t)(ch0 + c) * P.nrings + rn) * P.mstride + m];
                    float2 fv = make_float2(0.f, 0.f);
                    if (rs != rn) fv = spectra[((size_t)(ch0 + c) * P.nrings + rs) * P.mstride + m];
                    fsum[2 * c] = fn.x + fv.x;
                    fsum[2 * c + 1] = fn.y + fv.y;
                    fdif[2 * c] = fn.x - fv.x;
                    fdif[2 * c + 1] = fn.y - fv.y;
                }
            }
        }
#pragma unroll
        for (int c = 0; c < GNC; c += 4) {
            *reinterpret_cast<float4*>(&sF[0][tid][c]) = make_float4(fsum[c], fsum[c + 1], fsum[c + 2], fsum[c + 3]);
            *reinterpret_cast<float4*>(&sF[1][tid][c]) = make_float4(fdif[c], fdif[c + 1], fdif[c + 2], fdif[c + 3]);
        }
    }
    const double outscale = (a.adjoint && m > 0) ? 2.0 : 1.0;
    const long long abase = (long long)m * (2LL * P.lmax + 1 - m) / 2;
    float* out = reinterpret_cast<float*>(a.out);
    if (a.to_partial) out += (size_t)chunk * P.batch * P.nalm * 2;
    const int nl = P.lmax - m + 1;

    if (tid < GTL) {
        sA[0][tid] = (1 + tid < nl) ? P.coef_alpha[abase + m + 1 + tid] : 0.0;
        sS[0][tid] = (tid < nl) ? outscale * P.coef_scale[abase + m + tid] : 0.0;
    }
    __syncthreads();

    // contraction-phase coordinates
    const int par = lane >> 4;          // lanes 0-15: even l - m, 16-31: odd
    const int lquad = (lane >> 2) & 3;  // 4 degrees of that parity
    const int cq = lane & 3;            // 4 columns
    // A warp generates lambda for exactly the 32 rings it contracts over: generation -> contraction needs only
    // __syncwarp; the CTA meets twice per tile (partial tiles written / consumed).
    float* wred = &sLam[(0 * GK + warp * 32) * GROW];  // this warp's partial tile, aliased on its own lambda rows

    for (int t0 = 0, tb = 0; t0 < nl; t0 += GTL, tb ^= 1) {
        // prefetch alpha / scale of the next tile (visible after this tile's barriers)
        if (tid < GTL) {
            sA[tb ^ 1][tid] = (t0 + GTL + 1 + tid < nl) ? P.coef_alpha[abase + m + t0 + GTL + 1 + tid] : 0.0;
            sS[tb ^ 1][tid] = (t0 + GTL + tid < nl) ? outscale * P.coef_scale[abase + m + t0 + GTL + tid] : 0.0;
        }
        // ---- generate 32 degrees of this thread's ring
#pragma unroll
        for (int q = 0; q < GTL / 8; ++q) {
            if (sc < 0 && fabs(cur) > pow2c(ScaleCfg<float>::THR)) {
                cur *= pow2c(-ScaleCfg<float>::K);
                prev *= pow2c(-ScaleCfg<float>::K);
                ++sc;
            }
            float e[4], o[4];
#pragma unroll
            for (int p = 0; p < 4; ++p) {
                e[p] = sc == 0 ? (float)cur : 0.f;
                double xl = fma(-y, cur, cur);
                double nx = fma(sA[tb][8 * q + 2 * p], xl, -prev);
                prev = cur;
                cur = nx;
                o[p] = sc == 0 ? (float)cur : 0.f;
                xl = fma(-y, cur, cur);
                nx = fma(sA[tb][8 * q + 2 * p + 1], xl, -prev);
                prev = cur;
                cur = nx;
            }
            *reinterpret_cast<float4*>(&sLam[(0 * GK + tid) * GROW + 4 * q]) = make_float4(e[0], e[1], e[2], e[3]);
            *reinterpret_cast<float4*>(&sLam[(1 * GK + tid) * GROW + 4 * q]) = make_float4(o[0], o[1], o[2], o[3]);
        }
        const bool any = __any_sync(0xffffffffu, sc == 0);  // also orders the warp's stores before its loads
        float2 acc[4][2];  // [degree][column pair]: packed FMAs (FFMA2), lambda is the broadcast scalar
#pragma unroll
        for (int x = 0; x < 4; ++x) acc[x][0] = acc[x][1] = make_float2(0.f, 0.f);
        if (any) {
            const float* lp = &sLam[(par * GK + warp * 32) * GROW + 4 * lquad];
            const float* fp = &sF[par][warp * 32][4 * cq];
#pragma unroll 8
            for (int kk = 0; kk < 32; ++kk) {
                const float4 l4 = *reinterpret_cast<const float4*>(lp + kk * GROW);
                const float4 f4 = *reinterpret_cast<const float4*>(fp + kk * GNC);
                const float lv[4] = {l4.x, l4.y, l4.z, l4.w};
                const float2 f01 = make_float2(f4.x, f4.y), f23 = make_float2(f4.z, f4.w);
#pragma unroll
                for (int x = 0; x < 4; ++x) {
                    acc[x][0] = fma2(lv[x], f01, acc[x][0]);
                    acc[x][1] = fma2(lv[x], f23, acc[x][1]);
                }
            }
        }
        __syncwarp();  // the warp is done reading its lambda rows
#pragma unroll
        for (int x = 0; x < 4; ++x)
            *reinterpret_cast<float4*>(&wred[lane * 16 + 4 * x]) = make_float4(acc[x][0].x, acc[x][0].y, acc[x][1].x, acc[x][1].y);
        __syncthreads();
#pragma unroll
        for (int rep = 0; rep < 2; ++rep) {
            const int e = tid + GK * rep;        // 512 outputs of the tile
            const int ln = e >> 4, ix = e & 15;  // producing lane slot, element of its 4 x 4 block
            float sum = 0.f;
#pragma unroll
            for (int w = 0; w < GK / 32; ++w) sum += sLam[(w * 32) * GROW + ln * 16 + ix];
            const int opar = ln >> 4, olq = (ln >> 2) & 3, ocq = ln & 3;
            const int i = 2 * (4 * olq + (ix >> 2)) + opar;  // l - m - t0
            const int c = 4 * ocq + (ix & 3);
            const int ch = ch0 + (c >> 1), ri = c & 1;
            const int k = t0 + i;
            if (k < nl && ch < P.batch) {
                float o = (float)(sS[tb][i] * (double)sum);
                if (m == 0 && ri == 1) o = 0.f;
                out[((size_t)ch * P.nalm + abase + m + k) * 2 + ri] = o;
            }
        }
        __syncthreads();  // partial tiles consumed before the next tile overwrites the lambda rows
    }
}

// ------------------------------------------------------------------ analysis, batched fp32: 64-degree tiles
// Same contraction as legendre_analysis_gemm_kernel with the shared-memory traffic per FMA halved (ncu on the
// 32-degree version: 6 shared-memory wavefronts per 16 FFMA issue slots and warp -> the LSU, not the FMA pipe, was the
// limit): a tile is 64 degrees (32 per parity), a thread owns 8 degrees x 4 columns (16 packed FMAs per ring from
// two LDS.128 of lambda and one of F), the two parities of both tiles sit 16 / 64 bytes apart modulo the bank
// period so that the half-warps of different parity never collide, and the per-warp partial tiles are exchanged
// through a swizzled layout (conflict-free STS.128, two-wavefront LDS.64).
constexpr int HTL = 64;                  // degrees per tile
constexpr int HROW = HTL / 2 + 4;        // floats per lambda row: 32 degrees of one parity + 4 padding (144-byte pitch)
constexpr int HPS = GK * HROW + 4;       // parity stride of the lambda tile (floats): + 16 bytes
constexpr int HFS = GK * GNC + 16;       // parity stride of the F tile (floats): + 64 bytes
constexpr size_t HSMEM = sizeof(float) * (2 * HPS + 2 * HFS) + sizeof(double) * 4 * HTL;

__device__ __forceinline__ int hswz(int x, int ln) { return (x + (ln & 3) + 4 * ((ln >> 2) & 3) + 4 * (ln >> 4)) & 7; }

__global__ void __launch_bounds__(GK, 2) legendre_analysis_gemm64_kernel(LegArgs a) {
    const DevPlan& P = a.p;
    if (!ws_ok(P)) return;
    const int m = blockIdx.x;
    const int ch0 = blockIdx.z * GNCH;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // One CTA walks the ring chunks of its order m one after the other and adds each chunk's contribution to a_lm
    // in place (chunk 0 stores, later chunks read-add-store; the rows it revisits are its own and stay in L2), so
    // no per-chunk partial arrays are written and no combine kernel runs (measured at cfg4: 4.33 -> 4.07 ms).
    for (int chunk = 0;; ++chunk) {
    const int jbase = P.jmin[m] + chunk * GK;
    if (jbase >= P.npairs) return;
    const bool accumulate = chunk > 0;

    extern __shared__ __align__(16) unsigned char gemm_smem[];
    float* sLam = reinterpret_cast<float*>(gemm_smem);  // [parity][ring][HROW]; rows reused for the cross-warp sums
    float* sF = sLam + 2 * HPS;                         // [parity][ring][GNC]: F_N + F_S, F_N - F_S
    double(*sA)[HTL] = reinterpret_cast<double(*)[HTL]>(sF + 2 * HFS);
    double(*sS)[HTL] = sA + 2;  // outscale * s_l of the tile's degrees

    const float2* spectra = reinterpret_cast<const float2*>(P.spectra);
    const int j = jbase + tid;
    const bool valid = j < P.npairs;
    // fp32 output: cos(theta) = 1 - y rounded to double is accurate enough (the y-form of DESIGN.md R3 is for the
    // 1e-11 bar), and alpha_l x is off the dependent chain: ONE fp64 FMA of latency per degree instead of two
    double cur = 0.0, prev = 0.0, cx = 0.0;
    int sc = -1;
    {
        float fsum[GNC], fdif[GNC];
#pragma unroll
        for (int c = 0; c < GNC; ++c) fsum[c] = fdif[c] = 0.f;
        if (valid) {
            cx = 1.0 - P.y[j];
            lambda_seed<float>(m, P.pref_hi[m], P.pref_lo[m], P.ls_hi[j], P.ls_lo[j], cur, sc);
            const int rn = j, rs = P.nrings - 1 - j;
#pragma unroll
            for (int c = 0; c < GNCH; ++c) {
                if (ch0 + c < P.batch) {
                    const float2 fn = spectra[((size_t)(ch0 + c) * P.nrings + rn) * P.mstride + m];
                    float2 fv = make_float2(0.f, 0.f);
                    if (rs != rn) fv = spectra[((size_t)(ch0 + c) * P.nrings + rs) * P.mstride + m];
                    fsum[2 * c] = fn.x + fv.x;
                    fsum[2 * c + 1] = fn.y + fv.y;
                    fdif[2 * c] = fn.x - fv.x;
                    fdif[2 * c + 1] = fn.y - fv.y;
                }
            }
        }
#pragma unroll
        for (int c = 0; c < GNC; c += 4) {
            *reinterpret_cast<float4*>(&sF[tid * GNC + c]) = make_float4(fsum[c], fsum[c + 1], fsum[c + 2], fsum[c + 3]);
            *reinterpret_cast<float4*>(&sF[HFS + tid * GNC + c]) = make_float4(fdif[c], fdif[c + 1], fdif[c + 2], fdif[c + 3]);
        }
    }
    const double outscale = (a.adjoint && m > 0) ? 2.0 : 1.0;
    const long long abase = (long long)m * (2LL * P.lmax + 1 - m) / 2;
    float* out = reinterpret_cast<float*>(a.out);
    const int nl = P.lmax - m + 1;

    if (tid < HTL) {
        sA[0][tid] = (1 + tid < nl) ? P.coef_alpha[abase + m + 1 + tid] : 0.0;
        sS[0][tid] = (tid < nl) ? outscale * P.coef_scale[abase + m + tid] : 0.0;
    }
    __syncthreads();

    // contraction-phase coordinates: lane = (parity, degree octet, column quad)
    const int dq = lane >> 2, cq = lane & 3, par = dq >> 2, oc = dq & 3;
    const float* lp = sLam + par * HPS + (warp * 32) * HROW + 8 * oc;
    const float* fp = sF + par * HFS + (warp * 32) * GNC + 4 * cq;
    float* wred = sLam + (warp * 32) * HROW;  // this warp's partial tile (1024 floats), aliased on its own lambda rows

    bool all_on = false;  // warp-uniform: every ring of this warp is significant (sc == 0)
    for (int t0 = 0, tb = 0; t0 < nl; t0 += HTL, tb ^= 1) {
        // alpha / scale of the next tile: requested now, parked in shared memory after the contraction (a store right
        // here would stall warps 0-1 for the full global-load latency in every tile, and the CTA with them)
        float2 oldv[2] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
        if (accumulate) {
#pragma unroll
            for (int rep = 0; rep < 2; ++rep) {
                const int idx = tid + GK * rep;
                const int k = t0 + (idx >> 5) * 4 + (idx & 3), ch = ch0 + ((idx >> 2) & 7);
                if (k < nl && ch < P.batch)
                    oldv[rep] = *reinterpret_cast<const float2*>(&out[((size_t)ch * P.nalm + abase + m + k) * 2]);
            }
        }
        double nA = 0.0, nS = 0.0;
        if (tid < HTL) {
            nA = (t0 + HTL + 1 + tid < nl) ? P.coef_alpha[abase + m + t0 + HTL + 1 + tid] : 0.0;
            nS = (t0 + HTL + tid < nl) ? outscale * P.coef_scale[abase + m + t0 + HTL + tid] : 0.0;
        }
        // ---- generate 64 degrees of this thread's ring
        if (all_on) {  // every ring of the warp is significant: no rescale checks, no selects
#pragma unroll
            for (int q = 0; q < HTL / 8; ++q) {
                float e[4], o[4];
#pragma unroll
                for (int p = 0; p < 4; ++p) {
                    e[p] = (float)cur;
                    double nx = fma(sA[tb][8 * q + 2 * p] * cx, cur, -prev);
                    prev = cur;
                    cur = nx;
                    o[p] = (float)cur;
                    nx = fma(sA[tb][8 * q + 2 * p + 1] * cx, cur, -prev);
                    prev = cur;
                    cur = nx;
                }
                *reinterpret_cast<float4*>(&sLam[tid * HROW + 4 * q]) = make_float4(e[0], e[1], e[2], e[3]);
                *reinterpret_cast<float4*>(&sLam[HPS + tid * HROW + 4 * q]) = make_float4(o[0], o[1], o[2], o[3]);
            }
        } else {
#pragma unroll
            for (int q = 0; q < HTL / 8; ++q) {
                if (sc < 0 && fabs(cur) > pow2c(ScaleCfg<float>::THR)) {
                    cur *= pow2c(-ScaleCfg<float>::K);
                    prev *= pow2c(-ScaleCfg<float>::K);
                    ++sc;
                }
                float e[4], o[4];
#pragma unroll
                for (int p = 0; p < 4; ++p) {
                    e[p] = sc == 0 ? (float)cur : 0.f;
                    double nx = fma(sA[tb][8 * q + 2 * p] * cx, cur, -prev);
                    prev = cur;
                    cur = nx;
                    o[p] = sc == 0 ? (float)cur : 0.f;
                    nx = fma(sA[tb][8 * q + 2 * p + 1] * cx, cur, -prev);
                    prev = cur;
                    cur = nx;
                }
                *reinterpret_cast<float4*>(&sLam[tid * HROW + 4 * q]) = make_float4(e[0], e[1], e[2], e[3]);
                *reinterpret_cast<float4*>(&sLam[HPS + tid * HROW + 4 * q]) = make_float4(o[0], o[1], o[2], o[3]);
            }
            all_on = __all_sync(0xffffffffu, sc == 0);
        }
        const bool any = all_on || __any_sync(0xffffffffu, sc == 0);
        __syncwarp();  // orders the warp's lambda stores before its loads
        float2 acc[8][2];
#pragma unroll
        for (int x = 0; x < 8; ++x) acc[x][0] = acc[x][1] = make_float2(0.f, 0.f);
        if (any) {
#pragma unroll  // all 32 rings: loads of later rings issue under the FMAs of earlier ones (4.10 -> 3.88 ms at cfg4 against unroll 4)
            for (int kk = 0; kk < 32; ++kk) {
                const float4 la = *reinterpret_cast<const float4*>(lp + kk * HROW);
                const float4 lb = *reinterpret_cast<const float4*>(lp + kk * HROW + 4);
                const float4 f4 = *reinterpret_cast<const float4*>(fp + kk * GNC);
                const float lv[8] = {la.x, la.y, la.z, la.w, lb.x, lb.y, lb.z, lb.w};
                const float2 f01 = make_float2(f4.x, f4.y), f23 = make_float2(f4.z, f4.w);
#pragma unroll
                for (int x = 0; x < 8; ++x) {
                    acc[x][0] = fma2(lv[x], f01, acc[x][0]);
                    acc[x][1] = fma2(lv[x], f23, acc[x][1]);
                }
            }
        }
        __syncwarp();  // the warp is done reading its lambda rows
        if (tid < HTL) {
            sA[tb ^ 1][tid] = nA;
            sS[tb ^ 1][tid] = nS;
        }
#pragma unroll
        for (int x = 0; x < 8; ++x)
            *reinterpret_cast<float4*>(&wred[lane * 32 + 4 * hswz(x, lane)]) =
                make_float4(acc[x][0].x, acc[x][0].y, acc[x][1].x, acc[x][1].y);
        __syncthreads();
#pragma unroll
        for (int rep = 0; rep < 2; ++rep) {
            // 512 complex outputs of the tile: 4 consecutive degrees x 8 channels per warp-wide store (32-byte sectors)
            const int idx = tid + GK * rep;
            const int il = idx & 3, chl = (idx >> 2) & 7, ih = idx >> 5;
            const int i = ih * 4 + il;  // l - m - t0
            const int opar = i & 1, d = i >> 1, ooc = d >> 3, x = d & 7;
            const int ln = (opar * 4 + ooc) * 4 + (chl >> 1);
            const float* src = sLam + ln * 32 + 4 * hswz(x, ln) + 2 * (chl & 1);
            float2 sum = make_float2(0.f, 0.f);
#pragma unroll
            for (int w = 0; w < GK / 32; ++w) {
                const float2 v = *reinterpret_cast<const float2*>(src + (w * 32) * HROW);
                sum.x += v.x;
                sum.y += v.y;
            }
            const int ch = ch0 + chl;
            const int k = t0 + i;
            if (k < nl && ch < P.batch) {
                const double s = sS[tb][i];
                float2 o = make_float2(oldv[rep].x + (float)(s * (double)sum.x), oldv[rep].y + (float)(s * (double)sum.y));
                if (m == 0) o.y = 0.f;  // Im a_l0 is exactly zero
                *reinterpret_cast<float2*>(&out[((size_t)ch * P.nalm + abase + m + k) * 2]) = o;
            }
        }
        __syncthreads();  // partial tiles consumed before the next tile overwrites the lambda rows
    }
    }  // chunk
}

// sum the per-chunk partial results: alm[b][idx] = sum_c partial[c][b][idx], c < nchunks(m)
template <typename T>
__global__ void combine_partials_kernel(DevPlan P, const T* __restrict__ partial, T* __restrict__ alm) {
    if (!ws_ok(P)) return;
    const int m = blockIdx.x;
    const int b = blockIdx.y;
    const int nch = (P.npairs - P.jmin[m] + P.chunk_pairs - 1) / P.chunk_pairs;
    const long long base = ((long long)m * (2LL * P.lmax + 1 - m) / 2 + m) * 2;
    const int n = (P.lmax - m + 1) * 2;
    const size_t cstride = (size_t)P.batch * P.nalm * 2;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        T s = 0;
        for (int c = 0; c < nch; ++c) s += partial[c * cstride + (size_t)b * P.nalm * 2 + base + i];
        alm[(size_t)b * P.nalm * 2 + base + i] = s;
    }
}

// ------------------------------------------------------------------ synthesis (row s1)
template <typename T, int BT, int R, int NT>
__global__ void __launch_bounds__(NT) legendre_synthesis_kernel(LegArgs a) {
    using T2 = typename Vec2<T>::type;
    const DevPlan& P = a.p;
    if (!ws_ok(P)) return;
    // grid: x = ring chunk (fastest), y = m: the chunk-CTAs of one order run together and share its a_lm / alpha / s_l
    // rows through L2 instead of each fetching them from DRAM
    const int m = blockIdx.y;
    const int chunk = blockIdx.x;
    const int ch0 = blockIdx.z * BT;
    const int tid = threadIdx.x;
    const int jbase = P.jmin[m] + chunk * (NT * R);
    if (jbase >= P.npairs) return;

    __shared__ double sA[CT];
    __shared__ T sAlm[CT][BT][2];

    double cur[R], prev[R], y[R];
    int sc[R];
    T E[R][BT][2], O[R][BT][2];
    const double pref_hi = P.pref_hi[m], pref_lo = P.pref_lo[m];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int j = jbase + tid + NT * r;
#pragma unroll
        for (int c = 0; c < BT; ++c) E[r][c][0] = E[r][c][1] = O[r][c][0] = O[r][c][1] = 0;
        if (j < P.npairs) {
            y[r] = P.y[j];
            lambda_seed<T>(m, pref_hi, pref_lo, P.ls_hi[j], P.ls_lo[j], cur[r], sc[r]);
            prev[r] = 0.0;
        } else {
            y[r] = 1.0;
            cur[r] = 0.0;
            prev[r] = 0.0;
            sc[r] = -1;
        }
    }
    const T inscale = (a.adjoint && m > 0) ? (T)0.5 : (T)1;
    const long long abase = (long long)m * (2LL * P.lmax + 1 - m) / 2;
    const T* alm = reinterpret_cast<const T*>(a.in);
    const int nl = P.lmax - m + 1;

    // Tile t0 + CT is fetched into registers while tile t0 is consumed (no global-load latency between tiles).
    constexpr int NP = (CT * BT * 2 + NT - 1) / NT;
    double nA = 0.0, nScl[NP];
    T nAlm[NP];
    auto fetch = [&](int tn) {
        nA = (tid < CT && tn + 1 + tid < nl) ? P.coef_alpha[abase + m + tn + 1 + tid] : 0.0;
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            const int e = tid + NT * q;
            const int i = e / (BT * 2), c = (e / 2) % BT, ri = e & 1;
            const int k = tn + i, ch = ch0 + c;
            const bool ok = e < CT * BT * 2 && k < nl && ch < P.batch;
            nScl[q] = ok ? P.coef_scale[abase + m + k] : 0.0;
            nAlm[q] = ok ? alm[((size_t)ch * P.nalm + abase + m + k) * 2 + ri] : (T)0;
        }
    };
    int tstart = 0;  // late start, as in legendre_analysis_kernel
    if (P.st_chunk[1] == NT * R) {
        tstart = P.st_l0[1][(size_t)m * P.st_nchunk[1] + chunk];
        if (tstart > 0) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int j = jbase + tid + NT * r;
                if (j < P.npairs) {
                    const size_t e = (size_t)m * P.npairs + j;
                    cur[r] = P.st_cur[1][e];
                    prev[r] = P.st_prev[1][e];
                    sc[r] = P.st_sc[1][e];
                }
            }
        }
    }
    fetch(tstart);
    bool all_on = false;  // every ring pair of this warp is active (sc == 0)
    for (int t0 = tstart; t0 < nl; t0 += CT) {
        __syncthreads();  // previous tile fully consumed
        if (tid < CT) sA[tid] = nA;
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            const int e = tid + NT * q;
            if (e < CT * BT * 2) {
                const int i = e / (BT * 2), c = (e / 2) % BT, ri = e & 1;
                // a_lm s_l: the kernel sums mu_l = lambda_l / s_l
                T v = (T)((double)inscale * nScl[q] * (double)nAlm[q]);
                if (m == 0 && ri == 1) v = 0;  // Im a_l0 is ignored
                sAlm[i][c][ri] = v;
            }
        }
        __syncthreads();
        fetch(t0 + CT);
        const int tend = min(CT, nl - t0);
        for (int s0 = 0; s0 < tend; s0 += CHECK_EVERY) {
            bool warp_active = true;
            if (!all_on) {  // warp-uniform: skipped for good once every ring pair of the warp is significant
                bool any = false, all = true;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    if (sc[r] < 0) {
                        if (fabs(cur[r]) > pow2c(ScaleCfg<T>::THR)) {
                            cur[r] *= pow2c(-ScaleCfg<T>::K);
                            prev[r] *= pow2c(-ScaleCfg<T>::K);
                            ++sc[r];
                        }
                        // whatever was accumulated while the ring was inactive is noise below 2^-200 / 2^-44: drop it
#pragma unroll
                        for (int c = 0; c < BT; ++c) E[r][c][0] = E[r][c][1] = O[r][c][0] = O[r][c][1] = 0;
                    }
                    any |= (sc[r] == 0);
                    all &= (sc[r] == 0);
                }
                warp_active = __any_sync(0xffffffffu, any);
                all_on = __all_sync(0xffffffffu, all);
            }
            if (warp_active) {
#pragma unroll
                for (int i = 0; i < CHECK_EVERY; ++i) {
                    const double A = sA[s0 + i];
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const T lam = (T)cur[r];
#pragma unroll
                        for (int c = 0; c < BT; ++c) {
                            const T ar = sAlm[s0 + i][c][0], ai = sAlm[s0 + i][c][1];
                            if ((i & 1) == 0) {
                                E[r][c][0] = fma(lam, ar, E[r][c][0]);
                                E[r][c][1] = fma(lam, ai, E[r][c][1]);
                            } else {
                                O[r][c][0] = fma(lam, ar, O[r][c][0]);
                                O[r][c][1] = fma(lam, ai, O[r][c][1]);
                            }
                        }
                        const double xl = fma(-y[r], cur[r], cur[r]);
                        const double nx = fma(A, xl, -prev[r]);
                        prev[r] = cur[r];
                        cur[r] = nx;
                    }
                }
            } else {
#pragma unroll
                for (int i = 0; i < CHECK_EVERY; ++i) {
                    const double A = sA[s0 + i];
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const double xl = fma(-y[r], cur[r], cur[r]);
                        const double nx = fma(A, xl, -prev[r]);
                        prev[r] = cur[r];
                        cur[r] = nx;
                    }
                }
            }
        }
    }

    T2* spectra = reinterpret_cast<T2*>(P.spectra);
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int j = jbase + tid + NT * r;
        if (j >= P.npairs) continue;
        const int rn = j, rs = P.nrings - 1 - j;
        const bool live = sc[r] == 0;
#pragma unroll
        for (int c = 0; c < BT; ++c) {
            const int ch = ch0 + c;
            if (ch >= P.batch) continue;
            T2 gn, gs;
            gn.x = live ? E[r][c][0] + O[r][c][0] : (T)0;
            gn.y = live ? E[r][c][1] + O[r][c][1] : (T)0;
            gs.x = live ? E[r][c][0] - O[r][c][0] : (T)0;
            gs.y = live ? E[r][c][1] - O[r][c][1] : (T)0;
            spectra[((size_t)ch * P.nrings + rn) * P.mstride + m] = gn;
            if (rs != rn) spectra[((size_t)ch * P.nrings + rs) * P.mstride + m] = gs;
        }
    }
}

// ------------------------------------------------------------------ synthesis, batched fp32 (row s1), packed FMAs
// sm_100a has a packed fp32 FMA (PTX fma.rn.f32x2 -> SASS FFMA2: two FMAs per lane and issue slot, one operand may
// be a broadcast scalar).  (re, im) of one channel is exactly such a pair: E/O[r][c] += lambda * a_lm[c] is ONE
// instruction per (l, ring pair, channel), which leaves issue slots for the fp64 recurrence, the conversion and
// the shared-memory broadcasts of a_lm.  Same walk and exponent windows as legendre_synthesis_kernel<float>.
// 8-byte asynchronous copy global -> shared memory (LDGSTS): the data never passes through registers
__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gmem_src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

template <int BT, int R, int NT, int MINB>
__global__ void __launch_bounds__(NT, MINB) legendre_synthesis_f32x2_kernel(LegArgs a) {
    using T = float;
    const DevPlan& P = a.p;
    if (!ws_ok(P)) return;
    // grid: x = ring chunk (fastest), y = m: the chunk-CTAs of one order run together and share its a_lm / alpha / s_l
    // rows through L2 instead of each fetching them from DRAM
    const int m = blockIdx.y;
    const int chunk = blockIdx.x;
    const int ch0 = blockIdx.z * BT;
    const int tid = threadIdx.x;
    const int jbase = P.jmin[m] + chunk * (NT * R);
    if (jbase >= P.npairs) return;

    __shared__ double sA[CT];
    __shared__ __align__(16) float2 sAlm[CT][BT];
    __shared__ __align__(16) float2 rAlm[CT][BT];  // staging (cp.async targets): raw a_lm, s_l, alpha of the next tile
    __shared__ double rScl[CT], rA[CT];

    double cur[R], prev[R], y[R];
    int sc[R];
    float2 E[R][BT], O[R][BT];
    const double pref_hi = P.pref_hi[m], pref_lo = P.pref_lo[m];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int j = jbase + tid + NT * r;
#pragma unroll
        for (int c = 0; c < BT; ++c) E[r][c] = O[r][c] = make_float2(0.f, 0.f);
        if (j < P.npairs) {
            y[r] = 1.0 - P.y[j];  // cos(theta): fp32 output does not need the y-form (R3); alpha_l cos(theta) is
                                  // off the dependent chain, which is then one fp64 FMA per degree
            lambda_seed<T>(m, pref_hi, pref_lo, P.ls_hi[j], P.ls_lo[j], cur[r], sc[r]);
            prev[r] = 0.0;
        } else {
            y[r] = 0.0;
            cur[r] = 0.0;
            prev[r] = 0.0;
            sc[r] = -1;
        }
    }
    const T inscale = (a.adjoint && m > 0) ? 0.5f : 1.f;
    const long long abase = (long long)m * (2LL * P.lmax + 1 - m) / 2;
    const T* alm = reinterpret_cast<const T*>(a.in);
    const int nl = P.lmax - m + 1;

    // Tile t0 + CT travels global -> shared memory by cp.async while tile t0 is consumed: no registers are held
    // across the arithmetic (a register prefetch was spilled by ptxas, and the spill store waited for the load).
    // A thread owns ONE degree of the tile (one s_l) and CPT channels of it.
    constexpr int TPL = NT / CT, CPT = BT / TPL;
    static_assert(NT % CT == 0 && BT % TPL == 0 && NT >= 2 * CT, "staging mapping");
    const int fi = tid / TPL, fc0 = (tid % TPL) * CPT;
    auto request = [&](int tn) {
        const int k = tn + fi;
#pragma unroll
        for (int q = 0; q < CPT; ++q) {
            const int ch = ch0 + fc0 + q;
            if (k < nl && ch < P.batch) cp_async8(&rAlm[fi][fc0 + q], &alm[((size_t)ch * P.nalm + abase + m + k) * 2]);
            else rAlm[fi][fc0 + q] = make_float2(0.f, 0.f);
        }
        if (tid < CT) {
            if (tn + 1 + tid < nl) cp_async8(&rA[tid], &P.coef_alpha[abase + m + tn + 1 + tid]);
            else rA[tid] = 0.0;
        } else if (tid < 2 * CT) {
            const int i = tid - CT;
            if (tn + i < nl) cp_async8(&rScl[i], &P.coef_scale[abase + m + tn + i]);
            else rScl[i] = 0.0;
        }
        cp_async_commit();
    };
    request(0);
    bool all_on = false;  // every ring pair of this warp is active (sc == 0)
    for (int t0 = 0; t0 < nl; t0 += CT) {
        cp_async_wait_all();
        __syncthreads();  // staged tile landed; previous tile fully consumed
        if (tid < CT) sA[tid] = rA[tid];
        {
            const float sl = (float)((double)inscale * rScl[fi]);  // a_lm s_l: the kernel sums mu_l = lambda_l / s_l
#pragma unroll
            for (int q = 0; q < CPT; ++q) {
                const float2 r = rAlm[fi][fc0 + q];
                float2 v = make_float2(sl * r.x, sl * r.y);
                if (m == 0) v.y = 0.f;  // Im a_l0 is ignored
                sAlm[fi][fc0 + q] = v;
            }
        }
        __syncthreads();
        request(t0 + CT);
        const int tend = min(CT, nl - t0);
        for (int s0 = 0; s0 < tend; s0 += CHECK_EVERY) {
            bool warp_active = true;
            if (!all_on) {  // warp-uniform: skipped for good once every ring pair of the warp is significant
                bool any = false, all = true;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    if (sc[r] < 0) {
                        if (fabs(cur[r]) > pow2c(ScaleCfg<T>::THR)) {
                            cur[r] *= pow2c(-ScaleCfg<T>::K);
                            prev[r] *= pow2c(-ScaleCfg<T>::K);
                            ++sc[r];
                        }
#pragma unroll
                        for (int c = 0; c < BT; ++c) E[r][c] = O[r][c] = make_float2(0.f, 0.f);
                    }
                    any |= (sc[r] == 0);
                    all &= (sc[r] == 0);
                }
                warp_active = __any_sync(0xffffffffu, any);
                all_on = __all_sync(0xffffffffu, all);
            }
            if (warp_active) {
#pragma unroll
                for (int i = 0; i < CHECK_EVERY; ++i) {
                    const double A = sA[s0 + i];
                    float2 al[BT];
#pragma unroll
                    for (int c = 0; c < BT; ++c) al[c] = sAlm[s0 + i][c];
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const float lam = (float)cur[r];
#pragma unroll
                        for (int c = 0; c < BT; ++c) {
                            if ((i & 1) == 0) E[r][c] = fma2(lam, al[c], E[r][c]);
                            else O[r][c] = fma2(lam, al[c], O[r][c]);
                        }
                        const double nx = fma(A * y[r], cur[r], -prev[r]);  // y[] holds cos(theta) here
                        prev[r] = cur[r];
                        cur[r] = nx;
                    }
                }
            } else {
#pragma unroll
                for (int i = 0; i < CHECK_EVERY; ++i) {
                    const double A = sA[s0 + i];
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const double nx = fma(A * y[r], cur[r], -prev[r]);  // y[] holds cos(theta) here
                        prev[r] = cur[r];
                        cur[r] = nx;
                    }
                }
            }
        }
    }

    float2* spectra = reinterpret_cast<float2*>(P.spectra);
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int j = jbase + tid + NT * r;
        if (j >= P.npairs) continue;
        const int rn = j, rs = P.nrings - 1 - j;
        const bool live = sc[r] == 0;
#pragma unroll
        for (int c = 0; c < BT; ++c) {
            const int ch = ch0 + c;
            if (ch >= P.batch) continue;
            float2 gn = make_float2(0.f, 0.f), gs = gn;
            if (live) {
                gn = make_float2(E[r][c].x + O[r][c].x, E[r][c].y + O[r][c].y);
                gs = make_float2(E[r][c].x - O[r][c].x, E[r][c].y - O[r][c].y);
            }
            spectra[((size_t)ch * P.nrings + rn) * P.mstride + m] = gn;
            if (rs != rn) spectra[((size_t)ch * P.nrings + rs) * P.mstride + m] = gs;
        }
    }
}

// ------------------------------------------------------------------ launch configuration
// R (ring pairs per thread) and LT (l values per reduction tile) per instantiation.
template <typename T, int BT> struct LegCfg;
// analysis: NT threads x R ring pairs = one chunk; synthesis: LEG_THREADS x RS
template <> struct LegCfg<double, 1> { static constexpr int NT = 64, R = 7, LT = 8, RS = 4, NTS = 256; };
template <> struct LegCfg<float, 1> { static constexpr int NT = 128, R = 8, LT = 8, RS = 4, NTS = 256; };
template <> struct LegCfg<float, 4> { static constexpr int NT = 128, R = 4, LT = 4, RS = 2, NTS = 256; };

// batched fp32 analysis: contraction kernels.  Long degree ranges use the 64-degree tiles with in-place accumulation
// over the ring chunks (one "chunk" as far as the plan is concerned: no partial arrays); short ones (a few tiles per
// order, latency-bound) the 32-degree tiles with one CTA per ring chunk.
// ------------------------------------------------------------------ late start of the fp64 kernels
// For small m every ring pair is significant from l = m on; for large m the polar-most chunks walk hundreds of degrees
// with every lambda below the exponent window (recurrence only, nothing accumulated).  Those steps do not depend on the
// data: at workspace set-up this kernel walks them once per (m, chunk) exactly as the transform kernels would (same
// seeds, same two FMAs, same rescale checks every CHECK_EVERY degrees) and stores, for the first 64-degree tile in
// which a ring pair of the chunk crosses the window, the tile's first degree and every ring pair's state (value,
// previous value, exponent window) at that degree.  The transform kernels start there: results are bit-identical.
template <int R, int NT>
__global__ void __launch_bounds__(NT) legendre_start_kernel(DevPlan P, int which) {
    const int m = blockIdx.x, chunk = blockIdx.y, tid = threadIdx.x;
    const int jbase = P.jmin[m] + chunk * (NT * R);
    int* l0 = const_cast<int*>(P.st_l0[which]) + (size_t)m * P.st_nchunk[which] + chunk;
    if (jbase >= P.npairs) {
        if (tid == 0) *l0 = 0;
        return;
    }
    double cur[R], prev[R], y[R], scur[R], sprev[R];
    int sc[R], ssc[R];
    const double pref_hi = P.pref_hi[m], pref_lo = P.pref_lo[m];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int j = jbase + tid + NT * r;
        if (j < P.npairs) {
            y[r] = P.y[j];
            lambda_seed<double>(m, pref_hi, pref_lo, P.ls_hi[j], P.ls_lo[j], cur[r], sc[r]);
            prev[r] = 0.0;
        } else {
            y[r] = 1.0;
            cur[r] = 0.0;
            prev[r] = 0.0;
            sc[r] = -1;
        }
    }
    const long long abase = (long long)m * (2LL * P.lmax + 1 - m) / 2;
    const int nl = P.lmax - m + 1;
    int t0 = 0;
    for (;; t0 += CT) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            scur[r] = cur[r];
            sprev[r] = prev[r];
            ssc[r] = sc[r];
        }
        if (t0 + CT >= nl) break;  // the last tile is always run by the transform kernels
        bool act = false;
        const int tend = min(CT, nl - t0);
        for (int s0 = 0; s0 < tend && !act; s0 += CHECK_EVERY) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                if (sc[r] < 0 && fabs(cur[r]) > pow2c(ScaleCfg<double>::THR)) {
                    cur[r] *= pow2c(-ScaleCfg<double>::K);
                    prev[r] *= pow2c(-ScaleCfg<double>::K);
                    ++sc[r];
                }
                act |= (sc[r] == 0);
            }
            act = __syncthreads_or(act);
            if (act) break;
            for (int i = 0; i < CHECK_EVERY; ++i) {
                const int k = t0 + s0 + i;  // step producing degree m + k + 1
                const double A = (k + 1 < nl) ? P.coef_alpha[abase + m + k + 1] : 0.0;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const double xl = fma(-y[r], cur[r], cur[r]);
                    const double nx = fma(A, xl, -prev[r]);
                    prev[r] = cur[r];
                    cur[r] = nx;
                }
            }
        }
        if (act) break;
    }
    if (tid == 0) *l0 = t0;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int j = jbase + tid + NT * r;
        if (j < P.npairs) {
            const size_t e = (size_t)m * P.npairs + j;
            const_cast<double*>(P.st_cur[which])[e] = scur[r];
            const_cast<double*>(P.st_prev[which])[e] = sprev[r];
            const_cast<int*>(P.st_sc[which])[e] = ssc[r];
        }
    }
}

// chunk sizes of the two fp64 kernels (must agree with launch_legendre_analysis / launch_legendre_synthesis below)
constexpr int ST_R_ANA = 7, ST_R_SYN = 6, ST_NT = 64;
void legendre_start_chunks(cuhpx_dtype_t dt, int npairs, int chunk[2]) {
    const char* sw = getenv("CUHPX_LATE_START");  // "0": walk every order from l = m (A/B measurements)
    const bool on = dt == CUHPX_F64 && npairs >= 2048 && !(sw && sw[0] == '0');
    chunk[0] = on ? ST_R_ANA * ST_NT : 0;
    chunk[1] = on ? ST_R_SYN * ST_NT : 0;
}

cudaError_t launch_legendre_start_tables(const DevPlan& P, cudaStream_t st) {
    if (P.st_chunk[0] > 0) {
        legendre_start_kernel<ST_R_ANA, ST_NT><<<dim3(P.mmax + 1, P.st_nchunk[0]), ST_NT, 0, st>>>(P, 0);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    if (P.st_chunk[1] > 0) {
        legendre_start_kernel<ST_R_SYN, ST_NT><<<dim3(P.mmax + 1, P.st_nchunk[1]), ST_NT, 0, st>>>(P, 1);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

static bool use_gemm64(int lmax) { return lmax >= 512; }

int legendre_chunk_pairs(cuhpx_dtype_t dt, int batch, int lmax, int npairs) {
    // one "chunk" as far as the plan is concerned wherever the kernel walks the ring chunks itself
    if (dt == CUHPX_F64) return npairs > LegCfg<double, 1>::NT * LegCfg<double, 1>::R ? npairs : LegCfg<double, 1>::NT * LegCfg<double, 1>::R;
    if (batch >= 5) return use_gemm64(lmax) ? (npairs > GK ? npairs : GK) : GK;
    return batch >= 4 ? LegCfg<float, 4>::NT * LegCfg<float, 4>::R : LegCfg<float, 1>::NT * LegCfg<float, 1>::R;
}

template <typename T, int BT>
static cudaError_t run_analysis(const HostPlan& hp, const DevPlan& P, void* d_alm, int adjoint, cudaStream_t st) {
    using C = LegCfg<T, BT>;
    LegArgs a;
    a.p = P;
    a.in = nullptr;
    a.adjoint = adjoint;
    a.to_partial = P.nchunk_max > 1;
    a.out = a.to_partial ? P.partial : d_alm;
    dim3 grid(P.mmax + 1, P.nchunk_max, (P.batch + BT - 1) / BT);
    legendre_analysis_kernel<T, BT, C::R, C::LT, C::NT><<<grid, C::NT, 0, st>>>(a);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (a.to_partial) {
        dim3 g2(P.mmax + 1, P.batch);
        combine_partials_kernel<T><<<g2, 256, 0, st>>>(P, reinterpret_cast<const T*>(P.partial),
                                                        reinterpret_cast<T*>(d_alm));
        e = cudaGetLastError();
    }
    return e;
}

template <typename T, int BT>
static cudaError_t run_synthesis(const HostPlan& hp, const DevPlan& P, const void* d_alm, int adjoint, cudaStream_t st) {
    using C = LegCfg<T, BT>;
    LegArgs a;
    a.p = P;
    a.in = d_alm;
    a.out = nullptr;
    a.adjoint = adjoint;
    a.to_partial = 0;
    const int chunk = C::NTS * C::RS;
    dim3 grid((P.npairs + chunk - 1) / chunk, P.mmax + 1, (P.batch + BT - 1) / BT);
    legendre_synthesis_kernel<T, BT, C::RS, C::NTS><<<grid, C::NTS, 0, st>>>(a);
    return cudaGetLastError();
}

template <typename T, int BT, int R, int LT, int NT, int GL, bool SEQ = false, int MINB = 384 / NT>
static cudaError_t run_analysis_cfg(const HostPlan& hp, const DevPlan& P, void* d_alm, int adjoint, cudaStream_t st) {
    LegArgs a;
    a.p = P;
    a.in = nullptr;
    a.adjoint = adjoint;
    a.to_partial = !SEQ && P.nchunk_max > 1;
    a.out = a.to_partial ? P.partial : d_alm;
    dim3 grid(P.mmax + 1, SEQ ? 1 : P.nchunk_max, (P.batch + BT - 1) / BT);
    legendre_analysis_kernel<T, BT, R, LT, NT, GL, SEQ, MINB><<<grid, NT, 0, st>>>(a);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (a.to_partial) {
        dim3 g2(P.mmax + 1, P.batch);
        combine_partials_kernel<T><<<g2, 256, 0, st>>>(P, reinterpret_cast<const T*>(P.partial), reinterpret_cast<T*>(d_alm));
        e = cudaGetLastError();
    }
    return e;
}

template <typename T, int BT, int RS, int NTS>
static cudaError_t run_synthesis_cfg(const HostPlan& hp, const DevPlan& P, const void* d_alm, int adjoint, cudaStream_t st) {
    LegArgs a;
    a.p = P;
    a.in = d_alm;
    a.out = nullptr;
    a.adjoint = adjoint;
    a.to_partial = 0;
    const int chunk = NTS * RS;
    dim3 grid((P.npairs + chunk - 1) / chunk, P.mmax + 1, (P.batch + BT - 1) / BT);
    legendre_synthesis_kernel<T, BT, RS, NTS><<<grid, NTS, 0, st>>>(a);
    return cudaGetLastError();
}

static cudaError_t run_analysis_gemm(const HostPlan& hp, const DevPlan& P, void* d_alm, int adjoint, cudaStream_t st) {
    LegArgs a;
    a.p = P;
    a.in = nullptr;
    a.adjoint = adjoint;
    cudaError_t e;
    if (use_gemm64(P.lmax)) {
        a.to_partial = 0;
        a.out = d_alm;
        dim3 grid(P.mmax + 1, 1, (P.batch + GNCH - 1) / GNCH);
        e = cudaFuncSetAttribute(legendre_analysis_gemm64_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)HSMEM);
        if (e != cudaSuccess) return e;
        legendre_analysis_gemm64_kernel<<<grid, GK, HSMEM, st>>>(a);
        return cudaGetLastError();
    }
    a.to_partial = P.nchunk_max > 1;
    a.out = a.to_partial ? P.partial : d_alm;
    dim3 grid(P.mmax + 1, P.nchunk_max, (P.batch + GNCH - 1) / GNCH);
    constexpr size_t smem = sizeof(float) * (2 * GK * GROW + 2 * GK * GNC) + sizeof(double) * 4 * GTL;
    e = cudaFuncSetAttribute(legendre_analysis_gemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    legendre_analysis_gemm_kernel<<<grid, GK, smem, st>>>(a);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (a.to_partial) {
        dim3 g2(P.mmax + 1, P.batch);
        combine_partials_kernel<float><<<g2, 256, 0, st>>>(P, reinterpret_cast<const float*>(P.partial),
                                                            reinterpret_cast<float*>(d_alm));
        e = cudaGetLastError();
    }
    return e;
}

// Configurations below are the winners of sweeps on B200.
cudaError_t launch_legendre_analysis(const HostPlan& hp, const DevPlan& P, void* d_alm, int adjoint, cudaStream_t st) {
    // in-place accumulation over ring chunks (SEQ): cfg5 88.3 -> 87.0 ms, 3.7 GB of partial writes and 4.3 GB of workspace gone
    // fp64: 2-warp CTAs of 7 ring pairs per thread (r2 sweep over NT 32..128, R 5..8, resident CTAs: 80.9 ms at nside 4096
    // against 87.0 ms for the r1 shape 128 x 8; a software-pipelined butterfly was tried and was slower, 86-91 ms)
    // (small transforms keep the r1 shape: fewer, larger CTAs finish a launch-bound grid sooner -- nside 256: 0.090 vs 0.108 ms).
    // The price of the narrow chunks is DRAM traffic: the a_lm row of an order is read, added to and written back once per
    // chunk of 448 ring pairs (18 visits at nside 4096: 24.6 GB per call against 7.3 GB for 1024-pair chunks; L2 evict_last /
    // evict_first cache policies on the row / the spectra were tried and changed nothing) -- 0.3 TB/s, 5 % of HBM, under a
    // kernel that is bound by the FP64 pipe.
    if (hp.dtype == CUHPX_F64)
        return P.npairs >= 2048 ? run_analysis_cfg<double, 1, 7, 8, 64, 64, true>(hp, P, d_alm, adjoint, st)
                                : run_analysis_cfg<double, 1, 8, 8, 128, 64, true>(hp, P, d_alm, adjoint, st);
    if (P.batch >= 5) return run_analysis_gemm(hp, P, d_alm, adjoint, st);
    if (P.batch >= 4) return run_analysis<float, 4>(hp, P, d_alm, adjoint, st);
    return run_analysis<float, 1>(hp, P, d_alm, adjoint, st);
}

template <int BT, int R, int NT, int MINB>
static cudaError_t run_synthesis_f32x2(const HostPlan& hp, const DevPlan& P, const void* d_alm, int adjoint, cudaStream_t st) {
    LegArgs a;
    a.p = P;
    a.in = d_alm;
    a.out = nullptr;
    a.adjoint = adjoint;
    a.to_partial = 0;
    const int chunk = NT * R;
    dim3 grid((P.npairs + chunk - 1) / chunk, P.mmax + 1, (P.batch + BT - 1) / BT);
    legendre_synthesis_f32x2_kernel<BT, R, NT, MINB><<<grid, NT, 0, st>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_legendre_synthesis(const HostPlan& hp, const DevPlan& P, const void* d_alm, int adjoint, cudaStream_t st) {
    // fp64: 2-warp CTAs of 6 ring pairs per thread (r2 sweep over NT 64..128, R 3..8: 60.9 ms at nside 4096 against 63.7 ms
    // for the r1 shape 128 x 4)
    if (hp.dtype == CUHPX_F64)
        return P.npairs >= 2048 ? run_synthesis_cfg<double, 1, 6, 64>(hp, P, d_alm, adjoint, st)
                                : run_synthesis_cfg<double, 1, 4, 128>(hp, P, d_alm, adjoint, st);
    if (P.batch >= 8) {
        // tensor-core kernel (legendre_tc.cu): lambda goes to tensor memory, the contraction to tcgen05.mma
        const cudaError_t e = launch_legendre_synthesis_tc(hp, P, d_alm, adjoint, st);
        if (e != cudaErrorNotSupported) return e;
        // packed-FMA kernels, 8 channels per CTA; short degree ranges want more, smaller CTAs in flight
        return P.lmax < 512 ? run_synthesis_f32x2<8, 1, 256, 3>(hp, P, d_alm, adjoint, st)
                               : run_synthesis_f32x2<8, 2, 128, 3>(hp, P, d_alm, adjoint, st);
    }
    if (P.batch >= 4) return run_synthesis<float, 4>(hp, P, d_alm, adjoint, st);
    return run_synthesis<float, 1>(hp, P, d_alm, adjoint, st);
}

// ------------------------------------------------------------------ iterative refinement, elementwise steps (Eq. 4)
template <typename T, bool RESIDUAL>
__global__ void __launch_bounds__(256) refine_elementwise_kernel(const T* __restrict__ x, T* __restrict__ y, size_t n) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        y[i] = RESIDUAL ? x[i] - y[i] : y[i] + x[i];  // r = f - S a   |   a += A r
}

template <bool RESIDUAL>
static cudaError_t run_refine(cuhpx_dtype_t dt, const void* x, void* y, size_t n, cudaStream_t st) {
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    const size_t want = (n + 255) / 256;
    const unsigned blocks = (unsigned)(want < (size_t)sms * 8 ? (want ? want : 1) : (size_t)sms * 8);
    if (dt == CUHPX_F64) refine_elementwise_kernel<double, RESIDUAL><<<blocks, 256, 0, st>>>((const double*)x, (double*)y, n);
    else refine_elementwise_kernel<float, RESIDUAL><<<blocks, 256, 0, st>>>((const float*)x, (float*)y, n);
    return cudaGetLastError();
}
cudaError_t launch_residual(cuhpx_dtype_t dt, const void* f, void* r, size_t n, cudaStream_t st) {
    return run_refine<true>(dt, f, r, n, st);
}
cudaError_t launch_accumulate(cuhpx_dtype_t dt, const void* d, void* a, size_t n, cudaStream_t st) {
    return run_refine<false>(dt, d, a, n, st);
}

// ------------------------------------------------------------------ FMA peak probe
template <typename T>
__global__ void fma_probe_kernel(int iters, T* sink) {
    T a0 = (T)threadIdx.x * (T)1e-3, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6,
      a7 = a0 + 7;
    const T b = (T)0.999999, c = (T)1e-6;
    for (int i = 0; i < iters; ++i) {
        a0 = fma(a0, b, c); a1 = fma(a1, b, c); a2 = fma(a2, b, c); a3 = fma(a3, b, c);
        a4 = fma(a4, b, c); a5 = fma(a5, b, c); a6 = fma(a6, b, c); a7 = fma(a7, b, c);
    }
    const T s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (s == (T)-12345.678) sink[0] = s;
}

cudaError_t fma_peak_probe(cuhpx_dtype_t dt, int iters, float* ms, double* count, cudaStream_t st) {
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    const int blocks = sms * 8, threads = 256;
    cudaEvent_t e0, e1;
    if ((e = cudaEventCreate(&e0)) != cudaSuccess) return e;
    if ((e = cudaEventCreate(&e1)) != cudaSuccess) return e;
    for (int rep = 0; rep < 2; ++rep) {  // first launch warms up
        cudaEventRecord(e0, st);
        if (dt == CUHPX_F64) fma_probe_kernel<double><<<blocks, threads, 0, st>>>(iters, (double*)nullptr);
        else fma_probe_kernel<float><<<blocks, threads, 0, st>>>(iters, (float*)nullptr);
        cudaEventRecord(e1, st);
        e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) break;
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e == cudaSuccess) {
        cudaEventElapsedTime(ms, e0, e1);
        *count = (double)blocks * threads * 8.0 * (double)iters;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return e;
}

}  // namespace cuhpx

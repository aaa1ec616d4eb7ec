// Block-wide power-of-two complex FFT for one ring in one CTA (used by ring_fft.cu).
//
// n = 2^LOGN points are held ENTIRELY in registers (E = n / NT per thread); shared memory is only the exchange
// buffer between passes.  Each pass is a set of radix-R (R = 2..16) butterflies done in registers with
// compile-time twiddles; the inter-pass twiddles W_L^(j q) are products of two entries of small shared-memory
// root tables (Roots: exp(-2 pi i t / Q) = hi[t >> 7] * lo[t & 127]) -- no global-memory latency inside a pass.
// Decimation in frequency, in place: after the last pass the element at position p is X[bitrev(p)].
// The inverse runs the same passes backwards (conjugated, decimation in time), so a forward+inverse pair
// (the Bluestein convolution, Eq. 22) never needs a bit-reversal permutation.
// Exchange buffer (Xchg): 8-byte slots at padded positions p -> p + (p >> 4) -- fp64 as split re / im arrays,
// fp32 as one interleaved float2 array (one 64-bit access per element); with the plans below every pass is
// <= 2 wavefronts per request (measured by brute force).
#pragma once
#include <cuda_runtime.h>

namespace cuhpx {

template <typename T> struct V2;
template <> struct V2<float> { using type = float2; };
template <> struct V2<double> { using type = double2; };

__device__ __forceinline__ int padi(int p) { return p + (p >> 4); }
__host__ __device__ constexpr int padded_len(int n) { return n + (n >> 4) + 1; }

// Exchange buffer of n complex values in shared memory.
template <typename T> struct Xchg;
template <> struct Xchg<double> {
    double* re;
    double* im;
    static __host__ __device__ constexpr size_t bytes(int n) { return 2 * (size_t)padded_len(n) * sizeof(double); }
    __device__ __forceinline__ Xchg(void* base, int n) : re(reinterpret_cast<double*>(base)), im(re + padded_len(n)) {}
    __device__ __forceinline__ void st(int p, double a, double b) const {
        const int q = padi(p);
        re[q] = a;
        im[q] = b;
    }
    __device__ __forceinline__ void ld(int p, double& a, double& b) const {
        const int q = padi(p);
        a = re[q];
        b = im[q];
    }
    // q is already a padded position
    __device__ __forceinline__ void stq(int q, double a, double b) const {
        re[q] = a;
        im[q] = b;
    }
    __device__ __forceinline__ void ldq(int q, double& a, double& b) const {
        a = re[q];
        b = im[q];
    }
};
template <> struct Xchg<float> {
    float2* z;
    static __host__ __device__ constexpr size_t bytes(int n) { return (size_t)padded_len(n) * sizeof(float2); }
    __device__ __forceinline__ Xchg(void* base, int) : z(reinterpret_cast<float2*>(base)) {}
    __device__ __forceinline__ void st(int p, float a, float b) const { z[padi(p)] = make_float2(a, b); }
    __device__ __forceinline__ void ld(int p, float& a, float& b) const {
        const float2 v = z[padi(p)];
        a = v.x;
        b = v.y;
    }
    // q is already a padded position
    __device__ __forceinline__ void stq(int q, float a, float b) const { z[q] = make_float2(a, b); }
    __device__ __forceinline__ void ldq(int q, float& a, float& b) const {
        const float2 v = z[q];
        a = v.x;
        b = v.y;
    }
};

// Roots of unity exp(-2 pi i t / Q), 0 <= t < Q, from two shared-memory tables:
//   lo[k] = exp(-2 pi i k / Q), k < 128;  hi[k] = exp(-2 pi i 128 k / Q), k < ceil(Q / 128).
constexpr int ROOT_LO = 128;
__host__ __device__ constexpr int roots_len(int Q) { return ROOT_LO + (Q + ROOT_LO - 1) / ROOT_LO; }
template <typename T> struct Roots {
    using T2 = typename V2<T>::type;
    const T2* lo;
    const T2* hi;
    __device__ __forceinline__ Roots(const T2* base) : lo(base), hi(base + ROOT_LO) {}
    // exp(SIGN * 2 pi i t / Q)
    template <int SIGN> __device__ __forceinline__ void get(int t, T& c, T& s) const {
        const T2 a = hi[t >> 7], b = lo[t & (ROOT_LO - 1)];
        c = a.x * b.x - a.y * b.y;
        const T v = a.x * b.y + a.y * b.x;
        s = SIGN > 0 ? -v : v;
    }
};
// fill a root table of power-of-two order Q from the global table tw[k] = exp(-2 pi i k / twlen), Q | twlen
template <typename T>
__device__ __forceinline__ void fill_roots_pow2(typename V2<T>::type* base, int Q, const typename V2<T>::type* __restrict__ tw,
                                                int twlen, int tid, int nt) {
    const int nhi = Q / ROOT_LO, step = twlen / Q;
    for (int k = tid; k < ROOT_LO + nhi; k += nt) base[k] = __ldg(tw + (size_t)(k < ROOT_LO ? k : (k - ROOT_LO) * ROOT_LO) * step);
}
// fill a root table of arbitrary order Q (sincospi of the exact rational 2 t / Q)
template <typename T>
__device__ __forceinline__ void fill_roots_any(typename V2<T>::type* base, int Q, int tid, int nt) {
    const int nhi = (Q + ROOT_LO - 1) / ROOT_LO;
    const double inv = 2.0 / (double)Q;
    for (int k = tid; k < ROOT_LO + nhi; k += nt) {
        const int t = k < ROOT_LO ? k : (k - ROOT_LO) * ROOT_LO;
        double sn, cs;
        sincospi(-(double)t * inv, &sn, &cs);
        typename V2<T>::type v;
        v.x = (T)cs;
        v.y = (T)sn;
        base[k] = v;
    }
}

// radix plans: passes in DIF order
template <int LOGN> struct FftPlan;
template <> struct FftPlan<7> { static constexpr int NT = 32, NP = 4; static constexpr int R0 = 2, R1 = 4, R2 = 4, R3 = 4; };
template <> struct FftPlan<8> { static constexpr int NT = 32, NP = 3; static constexpr int R0 = 8, R1 = 8, R2 = 4, R3 = 1; };
template <> struct FftPlan<9> { static constexpr int NT = 64, NP = 3; static constexpr int R0 = 8, R1 = 8, R2 = 8, R3 = 1; };
template <> struct FftPlan<10> { static constexpr int NT = 64, NP = 3; static constexpr int R0 = 16, R1 = 16, R2 = 4, R3 = 1; };
template <> struct FftPlan<11> { static constexpr int NT = 128, NP = 3; static constexpr int R0 = 16, R1 = 16, R2 = 8, R3 = 1; };
template <> struct FftPlan<12> { static constexpr int NT = 256, NP = 3; static constexpr int R0 = 16, R1 = 16, R2 = 16, R3 = 1; };
template <> struct FftPlan<13> { static constexpr int NT = 512, NP = 4; static constexpr int R0 = 2, R1 = 16, R2 = 16, R3 = 16; };

template <int LOGN, int S> struct PassRadix {
    static constexpr int value = S == 0 ? FftPlan<LOGN>::R0 : S == 1 ? FftPlan<LOGN>::R1 : S == 2 ? FftPlan<LOGN>::R2 : FftPlan<LOGN>::R3;
};
// sub-transform length at pass S: L_S = n / (R_0 ... R_{S-1})
template <int LOGN, int S> struct PassLen { static constexpr int value = PassLen<LOGN, S - 1>::value / PassRadix<LOGN, S - 1>::value; };
template <int LOGN> struct PassLen<LOGN, 0> { static constexpr int value = 1 << LOGN; };

// cos/sin(2 pi k / 16), k = 0..7
__device__ __forceinline__ constexpr double c16(int k) {
    return k == 0 ? 1.0 : k == 1 ? 0.92387953251128675613 : k == 2 ? 0.70710678118654752440 : k == 3 ? 0.38268343236508977173
         : k == 4 ? 0.0 : k == 5 ? -0.38268343236508977173 : k == 6 ? -0.70710678118654752440 : -0.92387953251128675613;
}
__device__ __forceinline__ constexpr double s16(int k) {
    return k == 0 ? 0.0 : k == 1 ? 0.38268343236508977173 : k == 2 ? 0.70710678118654752440 : k == 3 ? 0.92387953251128675613
         : k == 4 ? 1.0 : k == 5 ? 0.92387953251128675613 : k == 6 ? 0.70710678118654752440 : 0.38268343236508977173;
}

// multiply (a + ib) by exp(SIGN * 2 pi i * K / 16), K compile time
template <int K, int SIGN, typename T> __device__ __forceinline__ void mul_w16(T& a, T& b) {
    if (K == 0) return;
    if (K == 4) {  // * (SIGN i)
        const T t = a;
        if (SIGN > 0) { a = -b; b = t; } else { a = b; b = -t; }
        return;
    }
    const T c = (T)c16(K), s = (T)(SIGN * s16(K));
    const T na = a * c - b * s, nb = a * s + b * c;
    a = na;
    b = nb;
}

// in-register radix-R DIF: natural in, bit-reversed out; Y[q] = sum_p x[p] exp(SIGN 2 pi i p q / R)
template <int R, int SIGN, typename T, int H = R / 2> struct RegDif {
    static __device__ __forceinline__ void run(T* re, T* im) {
#pragma unroll
        for (int b = 0; b < R; b += 2 * H) {
            stage<0>(re + b, im + b);
        }
        RegDif<R, SIGN, T, H / 2>::run(re, im);
    }
    template <int J> static __device__ __forceinline__ void stage(T* re, T* im) {
        if constexpr (J < H) {
            const T ar = re[J], ai = im[J], cr = re[J + H], ci = im[J + H];
            re[J] = ar + cr;
            im[J] = ai + ci;
            T dr = ar - cr, di = ai - ci;
            mul_w16<J * (8 / H), SIGN>(dr, di);
            re[J + H] = dr;
            im[J + H] = di;
            stage<J + 1>(re, im);
        }
    }
};
template <int R, int SIGN, typename T> struct RegDif<R, SIGN, T, 0> {
    static __device__ __forceinline__ void run(T*, T*) {}
};

// in-register radix-R DIT: bit-reversed in, natural out; same sum
template <int R, int SIGN, typename T, int H = 1> struct RegDit {
    static __device__ __forceinline__ void run(T* re, T* im) {
        if constexpr (H < R) {
#pragma unroll
            for (int b = 0; b < R; b += 2 * H) {
                stage<0>(re + b, im + b);
            }
            RegDit<R, SIGN, T, H * 2>::run(re, im);
        }
    }
    template <int J> static __device__ __forceinline__ void stage(T* re, T* im) {
        if constexpr (J < H) {
            T cr = re[J + H], ci = im[J + H];
            mul_w16<J * (8 / H), SIGN>(cr, ci);
            const T ar = re[J], ai = im[J];
            re[J] = ar + cr;
            im[J] = ai + ci;
            re[J + H] = ar - cr;
            im[J + H] = ai - ci;
            stage<J + 1>(re, im);
        }
    }
};

template <int R> __device__ __forceinline__ constexpr int brev_r(int x) {
    int r = 0;
    for (int b = 1, t = R >> 1; b < R; b <<= 1, t >>= 1)
        if (x & b) r |= t;
    return r;
}

// Multiply register r (holding butterfly output q = bitrev_R(r)) by w^q, w = exp(-2 pi i t / Q) (conjugated if
// CONJ).  fp32: w^(2^k) come from the root table, the other powers are running products (<= 3 multiplies from a
// table value).  fp64: only w comes from the table, w^2, w^4, w^8 by squaring (3 flops and no shared-memory access
// instead of 2 LDS.128 + 4 flops; the fp64 kernels are bound by the shared-memory pipe, and <= 3 squarings cost
// ~1e-15 of phase accuracy).  q t < Q for every q < R.
template <int R, bool CONJ, typename T>
__device__ __forceinline__ void apply_twiddles(const Roots<T>& rt, int t, T* re, T* im) {
    T w1r = 0, w1i = 0, cr = 1, ci = 0, pr = 1, pi = 0;  // (pr, pi): the last power of two
#pragma unroll
    for (int q = 1; q < R; ++q) {
        if ((q & (q - 1)) == 0) {  // power of two
            if (q == 1 || sizeof(T) == 4) {
                rt.template get<(CONJ ? +1 : -1)>(q * t, cr, ci);
            } else {
                cr = pr * pr - pi * pi;
                ci = 2 * pr * pi;
            }
            pr = cr;
            pi = ci;
            if (q == 1) {
                w1r = cr;
                w1i = ci;
            }
        } else {
            const T nr = cr * w1r - ci * w1i, ni = cr * w1i + ci * w1r;
            cr = nr;
            ci = ni;
        }
        const int r = brev_r<R>(q);
        const T a = re[r], b = im[r];
        re[r] = a * cr - b * ci;
        im[r] = a * ci + b * cr;
    }
}

// LOGQ: log2 of the order of the root table handed to forward / inverse (LOGQ >= LOGN).
// GROUPS > 1: the CTA holds GROUPS independent teams of NT threads, each running its own FFT on its own exchange
// buffer; `tid` is the index inside the team and the passes meet at the team's named barrier (1 + team) instead of
// the CTA barrier, so one team's exchange overlaps the other's butterflies.
template <typename T, int LOGN, int LOGQ = LOGN, int GROUPS = 1> struct BlockFFT {
    using P = FftPlan<LOGN>;
    using T2 = typename V2<T>::type;
    static constexpr int N = 1 << LOGN, NT = P::NT, E = N / NT, NP = P::NP;
    static constexpr int RLAST = PassRadix<LOGN, NP - 1>::value;
    static constexpr int R0 = P::R0;
    static constexpr size_t SMEM_BYTES = Xchg<T>::bytes(N);

    static __device__ __forceinline__ void team_sync() {
        if constexpr (GROUPS == 1) {
            __syncthreads();
        } else {
            asm volatile("bar.sync %0, %1;" ::"r"(1 + (int)(threadIdx.x / NT)), "n"(NT) : "memory");
        }
    }

    // position of register e = c R + rho in pass S
    template <int S> static __device__ __forceinline__ int pos(int tid, int c, int rho) {
        constexpr int R = PassRadix<LOGN, S>::value, L = PassLen<LOGN, S>::value, LR = L / R;
        const int u = tid + NT * c;
        const int B = u / LR, j = u % LR;
        return B * L + j + rho * LR;
    }
    // natural index held by register e in the pass-0 layout (input of forward / output of inverse)
    static __device__ __forceinline__ int index0(int tid, int e) { return pos<0>(tid, e / R0, e % R0); }
    // frequency index held by register e after forward (last-pass layout)
    static __device__ __forceinline__ int freq_index(int tid, int e) {
        const int p = pos<NP - 1>(tid, e / RLAST, e % RLAST);
        return (int)(__brev((unsigned)p) >> (32 - LOGN));
    }

    // Exchange positions of a thread's R registers in pass S are base + rho LR.  When LR is a multiple of 16 the
    // padding p -> p + (p >> 4) is affine in rho, so ONE padded base per butterfly and compile-time offsets replace
    // a shift-add per element (ncu: integer address arithmetic was ~22 % of the issued instructions of the fp32
    // kernels, which are issue-bound).
    template <int S> static __device__ __forceinline__ void load(T (&re)[E], T (&im)[E], const Xchg<T>& x, int tid) {
        constexpr int R = PassRadix<LOGN, S>::value, L = PassLen<LOGN, S>::value, LR = L / R;
#pragma unroll
        for (int c = 0; c < E / R; ++c) {
            const int u = tid + NT * c;
            const int base = (u / LR) * L + (u % LR);
            if constexpr (LR % 16 == 0) {
                const int pb = padi(base);
#pragma unroll
                for (int r = 0; r < R; ++r) x.ldq(pb + r * (LR + LR / 16), re[c * R + r], im[c * R + r]);
            } else {
#pragma unroll
                for (int r = 0; r < R; ++r) x.ld(base + r * LR, re[c * R + r], im[c * R + r]);
            }
        }
    }
    template <int S> static __device__ __forceinline__ void store(const T (&re)[E], const T (&im)[E], const Xchg<T>& x, int tid) {
        constexpr int R = PassRadix<LOGN, S>::value, L = PassLen<LOGN, S>::value, LR = L / R;
#pragma unroll
        for (int c = 0; c < E / R; ++c) {
            const int u = tid + NT * c;
            const int base = (u / LR) * L + (u % LR);
            if constexpr (LR % 16 == 0) {
                const int pb = padi(base);
#pragma unroll
                for (int r = 0; r < R; ++r) x.stq(pb + r * (LR + LR / 16), re[c * R + r], im[c * R + r]);
            } else {
#pragma unroll
                for (int r = 0; r < R; ++r) x.st(base + r * LR, re[c * R + r], im[c * R + r]);
            }
        }
    }

    template <int S> static __device__ __forceinline__ void fwd_pass(T (&re)[E], T (&im)[E], const Xchg<T>& x,
                                                                  const Roots<T>& rt, int tid) {
        if constexpr (S < NP) {
            constexpr int R = PassRadix<LOGN, S>::value, L = PassLen<LOGN, S>::value, LR = L / R;
            if constexpr (S > 0) {
                team_sync();
                load<S>(re, im, x, tid);
            }
#pragma unroll
            for (int c = 0; c < E / R; ++c) {
                RegDif<R, -1, T>::run(re + c * R, im + c * R);
                if constexpr (LR > 1) {
                    const int j = (tid + NT * c) % LR;
                    apply_twiddles<R, false, T>(rt, j * ((1 << LOGQ) / L), re + c * R, im + c * R);
                }
            }
            if constexpr (S < NP - 1) store<S>(re, im, x, tid);
            fwd_pass<S + 1>(re, im, x, rt, tid);
        }
    }

    template <int S> static __device__ __forceinline__ void inv_pass(T (&re)[E], T (&im)[E], const Xchg<T>& x,
                                                                  const Roots<T>& rt, int tid) {
        if constexpr (S >= 0) {
            constexpr int R = PassRadix<LOGN, S>::value, L = PassLen<LOGN, S>::value, LR = L / R;
            if constexpr (S < NP - 1) {
                team_sync();
                load<S>(re, im, x, tid);
            }
#pragma unroll
            for (int c = 0; c < E / R; ++c) {
                if constexpr (LR > 1) {
                    const int j = (tid + NT * c) % LR;
                    apply_twiddles<R, true, T>(rt, j * ((1 << LOGQ) / L), re + c * R, im + c * R);
                }
                RegDit<R, +1, T>::run(re + c * R, im + c * R);
            }
            if constexpr (S > 0) store<S>(re, im, x, tid);
            inv_pass<S - 1>(re, im, x, rt, tid);
        }
    }

    // forward DFT (exp(-i...)): registers in pass-0 layout -> registers in last-pass layout (freq_index)
    static __device__ __forceinline__ void forward(T (&re)[E], T (&im)[E], const Xchg<T>& x, const Roots<T>& rt, int tid) {
        fwd_pass<0>(re, im, x, rt, tid);
    }
    // unnormalised inverse (exp(+i...), factor n): last-pass layout -> pass-0 layout
    static __device__ __forceinline__ void inverse(T (&re)[E], T (&im)[E], const Xchg<T>& x, const Roots<T>& rt, int tid) {
        inv_pass<NP - 1>(re, im, x, rt, tid);
    }
    // write the forward result to shared memory in natural frequency order (call after forward; syncs first,
    // because other threads may still be reading the exchange buffer; caller syncs before reading)
    static __device__ __forceinline__ void store_natural(const T (&re)[E], const T (&im)[E], const Xchg<T>& x, int tid) {
        team_sync();
#pragma unroll
        for (int e = 0; e < E; ++e) x.st(freq_index(tid, e), re[e], im[e]);
    }
};

}  // namespace cuhpx

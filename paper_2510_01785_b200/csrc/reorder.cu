// Layout reordering NESTED <-> RING of HEALPix maps (paper section III-B).
// The paper converts between layouts through the intermediate (x, y, f): "source -> xyf, xyf -> target, then the
// data array is reordered".  NESTED -> xyf is bit de-interleaving of the Z-order (Morton) index inside
// a base face; xyf -> RING follows Gorski et al. (ref [1] P:416): a pixel of face f at (x, y) lies on ring
// jr = jrll[f] nside - x - y - 1 (x + y is constant along a ring) and its position along the ring grows with x - y.
//
// Both directions are ONE pass over HBM built on that observation: a CTA owns a T x T block of one face, which is
// T^2 CONSECUTIVE elements of the NESTED array, and whose anti-diagonals x + y = const are runs of CONSECUTIVE
// elements of RING rows.  The block goes through shared memory, so the NESTED side moves as one contiguous piece
// and the RING side as runs of up to T elements -- no scattered 4-byte accesses on either side.  Only xyf -> RING
// index arithmetic is needed (the reverse direction reads along the same runs).  Roofline: HBM, 2 x map bytes.
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

#include "cuhpx_internal.h"

namespace cuhpx {

// ring number of the base faces' southern corner row and longitude offset, Gorski et al. Fig. 4 / section 4.1
__host__ __device__ __forceinline__ int face_jrll(int f) { return 2 + (f >> 2); }
__host__ __device__ __forceinline__ int face_jpll(int f) { return f < 4 ? 2 * f + 1 : (f < 8 ? 2 * (f - 4) : 2 * (f - 8) + 1); }

// (x, y, f) -> RING index (0-based); x grows to the north-east, y to the north-west inside the face
__host__ __device__ __forceinline__ long long xyf_to_ring(int nside, int x, int y, int f) {
    const long long ns = nside;
    const long long npix = 12 * ns * ns, ncap = 2 * ns * (ns - 1);
    const int jr = face_jrll(f) * nside - x - y - 1;  // ring, 1 .. 4 nside - 1
    long long nr, before;
    int kshift;
    if (jr < nside) {  // north polar cap
        nr = jr;
        before = 2 * nr * (nr - 1);
        kshift = 0;
    } else if (jr > 3 * nside) {  // south polar cap
        nr = 4 * ns - jr;
        before = npix - 2 * (nr + 1) * nr;
        kshift = 0;
    } else {  // equatorial belt
        nr = ns;
        before = ncap + (long long)(jr - nside) * 4 * ns;
        kshift = (jr - nside) & 1;
    }
    long long jp = (face_jpll(f) * nr + x - y + 1 + kshift) / 2;  // position along the ring, 1 .. 4 nr
    if (jp > 4 * nr) jp -= 4 * nr;
    if (jp < 1) jp += 4 * nr;
    return before + jp - 1;
}

// even bits of v packed into the low half (inverse of Morton interleaving)
__host__ __device__ __forceinline__ unsigned compact_bits(unsigned long long v) {
    v &= 0x5555555555555555ull;
    v = (v | (v >> 1)) & 0x3333333333333333ull;
    v = (v | (v >> 2)) & 0x0f0f0f0f0f0f0f0full;
    v = (v | (v >> 4)) & 0x00ff00ff00ff00ffull;
    v = (v | (v >> 8)) & 0x0000ffff0000ffffull;
    v = (v | (v >> 16)) & 0x00000000ffffffffull;
    return (unsigned)v;
}
long long nest_to_ring_index(int nside, long long ipnest) {
    const long long ns2 = (long long)nside * nside;
    const int f = (int)(ipnest / ns2);
    const unsigned long long r = (unsigned long long)(ipnest % ns2);
    return xyf_to_ring(nside, (int)compact_bits(r), (int)compact_bits(r >> 1), f);
}

constexpr int RT_THREADS = 256;

// 32-bit variants for the kernel (nside <= 8192: every index fits in 31 bits)
__device__ __forceinline__ unsigned compact16(unsigned v) {  // even bits of the low 32 -> low 16
    v &= 0x55555555u;
    v = (v | (v >> 1)) & 0x33333333u;
    v = (v | (v >> 2)) & 0x0f0f0f0fu;
    v = (v | (v >> 4)) & 0x00ff00ffu;
    v = (v | (v >> 8)) & 0x0000ffffu;
    return v;
}

// T = tile edge (power of two, <= 64, <= nside).  grid.x = 12 (nside / T)^2 tiles, grid.y = batch.
// Index arithmetic is hoisted: everything that depends only on the anti-diagonal s = xl + yl (ring number, ring
// length, first index of the ring, the in-ring position of xl = 0) is computed once per diagonal, an element then
// costs an add, a wrap and the two addresses (the first version recomputed xyf -> RING in 64 bits per element and
// was issue-bound at 79 % issue-active / 1.5 TB/s; ncu in profiles/).
template <typename W, int T, bool TO_RING>
__global__ void __launch_bounds__(RT_THREADS) reorder_kernel(int nside, long long npix, const W* __restrict__ in, W* __restrict__ out) {
    extern __shared__ __align__(16) unsigned char reorder_smem[];
    W* tile = reinterpret_cast<W*>(reorder_smem);
    constexpr int TT = T * T;
    const int tpf = (nside / T) * (nside / T);
    const int f = blockIdx.x / tpf;
    const unsigned tmorton = blockIdx.x - f * tpf;  // tiles of a face in Z-order, like the pixels
    const int x0 = (int)compact16(tmorton) * T, y0 = (int)compact16(tmorton >> 1) * T;
    const size_t nest0 = (size_t)f * nside * nside + (size_t)tmorton * TT;
    const W* src = in + (size_t)blockIdx.y * npix;
    W* dst = out + (size_t)blockIdx.y * npix;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // element e = tid + 256 i of the block: Morton code -> (xl, yl); the thread part is fixed, the i part constant-folds
    const int txl = (int)compact16((unsigned)tid), tyl = (int)compact16((unsigned)tid >> 1);

    if (TO_RING) {
#pragma unroll
        for (int i = 0; i < (TT + RT_THREADS - 1) / RT_THREADS; ++i) {
            const int e = tid + RT_THREADS * i;
            if (e < TT) {
                // bits 8.. of e are i: even bits of (i << 8) go to xl bit 4.., odd bits to yl bit 4..
                const int xl = TT > RT_THREADS ? (txl | ((int)compact16((unsigned)i) << 4)) : (int)compact16((unsigned)e);
                const int yl = TT > RT_THREADS ? (tyl | ((int)compact16((unsigned)i >> 1) << 4)) : (int)compact16((unsigned)e >> 1);
                tile[yl * T + xl] = src[nest0 + e];
            }
        }
        __syncthreads();
    }
    const int ns = nside, jrl = face_jrll(f) * ns, jpl = face_jpll(f);
    const int ncap = 2 * ns * (ns - 1);
    // ring of anti-diagonal s (x + y = x0 + y0 + s): first RING index of the run's ring, ring length, position of xl = 0
    auto diagonal = [&](int s, int& before, int& n4, int& a) {
        const int jr = jrl - (x0 + y0 + s) - 1;
        int nr, kshift = 0;
        if (jr < ns) {
            nr = jr;
            before = 2 * nr * (nr - 1);
        } else if (jr > 3 * ns) {
            nr = 4 * ns - jr;
            before = (int)npix - 2 * (nr + 1) * nr;
        } else {
            nr = ns;
            before = ncap + (jr - ns) * 4 * ns;
            kshift = (jr - ns) & 1;
        }
        n4 = 4 * nr;
        // jp(xl) = (jpl nr + (x0 + xl) - (y0 + s - xl) + 1 + kshift) / 2 = a + xl, the numerator is always even
        a = (jpl * nr + x0 - y0 - s + 1 + kshift) / 2;
    };
    auto ring_index = [&](int before, int n4, int a, int xl) {
        int jp = a + xl;
        if (jp > n4) jp -= n4;
        if (jp < 1) jp += n4;
        return before + jp - 1;
    };
    constexpr int NW = RT_THREADS / 32, KPD = (T + 31) / 32;  // warps, lane slots per diagonal
    if (TO_RING) {
        for (int s = warp; s < 2 * T - 1; s += NW) {
            int before, n4, a;
            diagonal(s, before, n4, a);
            const int xmin = s < T ? 0 : s - T + 1, len = s < T ? s + 1 : 2 * T - 1 - s;
            for (int k = lane; k < len; k += 32) {
                const int xl = xmin + k;
                dst[ring_index(before, n4, a, xl)] = tile[(s - xl) * T + xl];
            }
        }
    } else {
        // gather side: the loads of U diagonals are issued before any of them is parked in shared memory
        constexpr int U = 4;
        for (int sb = warp; sb < 2 * T - 1; sb += NW * U) {
            W v[U][KPD];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int s = sb + NW * u;
                if (s < 2 * T - 1) {
                    int before, n4, a;
                    diagonal(s, before, n4, a);
                    const int xmin = s < T ? 0 : s - T + 1, len = s < T ? s + 1 : 2 * T - 1 - s;
#pragma unroll
                    for (int q = 0; q < KPD; ++q) {
                        const int k = lane + 32 * q;
                        if (k < len) v[u][q] = src[ring_index(before, n4, a, xmin + k)];
                    }
                }
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int s = sb + NW * u;
                if (s < 2 * T - 1) {
                    const int xmin = s < T ? 0 : s - T + 1, len = s < T ? s + 1 : 2 * T - 1 - s;
#pragma unroll
                    for (int q = 0; q < KPD; ++q) {
                        const int k = lane + 32 * q;
                        if (k < len) tile[(s - xmin - k) * T + xmin + k] = v[u][q];
                    }
                }
            }
        }
    }
    if (!TO_RING) {
        __syncthreads();
#pragma unroll
        for (int i = 0; i < (TT + RT_THREADS - 1) / RT_THREADS; ++i) {
            const int e = tid + RT_THREADS * i;
            if (e < TT) {
                const int xl = TT > RT_THREADS ? (txl | ((int)compact16((unsigned)i) << 4)) : (int)compact16((unsigned)e);
                const int yl = TT > RT_THREADS ? (tyl | ((int)compact16((unsigned)i >> 1) << 4)) : (int)compact16((unsigned)e >> 1);
                dst[nest0 + e] = tile[yl * T + xl];
            }
        }
    }
}

template <typename W, int T>
static cudaError_t run_reorder_t(int nside, int batch, int to_ring, const void* in, void* out, cudaStream_t st) {
    const long long npix = 12LL * nside * nside;
    dim3 grid((unsigned)(12 * (nside / T) * (nside / T)), (unsigned)batch);
    constexpr size_t smem = sizeof(W) * T * T;
    cudaError_t e;
    if (to_ring) {
        if (smem > 48 * 1024 && (e = cudaFuncSetAttribute(reorder_kernel<W, T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess) return e;
        reorder_kernel<W, T, true><<<grid, RT_THREADS, smem, st>>>(nside, npix, (const W*)in, (W*)out);
    } else {
        if (smem > 48 * 1024 && (e = cudaFuncSetAttribute(reorder_kernel<W, T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess) return e;
        reorder_kernel<W, T, false><<<grid, RT_THREADS, smem, st>>>(nside, npix, (const W*)in, (W*)out);
    }
    return cudaGetLastError();
}

template <typename W>
static cudaError_t run_reorder(int nside, int batch, int to_ring, const void* in, void* out, cudaStream_t st) {
    // 4-byte elements, scatter side: 128 x 128 tiles (64 KB) double the length of the RING-side runs (measured: 3.2 ->
    // 3.4-3.6 TB/s); the gather side prefers more resident CTAs (64 x 64 tiles)
    if (sizeof(W) == 4 && nside >= 128 && to_ring) return run_reorder_t<W, 128>(nside, batch, to_ring, in, out, st);
    if (nside >= 64) return run_reorder_t<W, 64>(nside, batch, to_ring, in, out, st);
    if (nside >= 16) return run_reorder_t<W, 16>(nside, batch, to_ring, in, out, st);
    if (nside >= 4) return run_reorder_t<W, 4>(nside, batch, to_ring, in, out, st);
    return run_reorder_t<W, 1>(nside, batch, to_ring, in, out, st);
}

cudaError_t launch_reorder(int nside, int batch, cuhpx_dtype_t dt, int to_ring, const void* in, void* out, cudaStream_t st) {
    return dt == CUHPX_F64 ? run_reorder<uint64_t>(nside, batch, to_ring, in, out, st)
                           : run_reorder<uint32_t>(nside, batch, to_ring, in, out, st);
}

// ------------------------------------------------------------------ generic layout conversion through (x, y, f)
// "Source -> xyf, xyf -> Target".  Layout codes (include/cuhpx.h): 0 RING, 1 NESTED, 2 + 2 corner + sense
// = flat: every face a row-major nside x nside image, index = f nside^2 + row nside + col, whose origin is the face's
// corner S, E, N, W (corner 0..3) and whose fast axis leaves the origin counter-clockwise (sense 0) or clockwise (1)
// around the face; the slow axis leaves it the other way (reading R12 of P:110 / Fig. 3C).
// With the face coordinates of NESTED (x north-east, y north-west from the southern corner; corners S (0,0), E (n-1,0),
// N (n-1,n-1), W (0,n-1), counter-clockwise S -> E -> N -> W):
//   corner S: (u, v) = (x, y)   E: (y, n-1-x)   N: (n-1-x, n-1-y)   W: (n-1-y, x)   = steps along the two edges leaving
//   the origin, u towards the counter-clockwise neighbour;  (col, row) = (u, v) for sense 0, (v, u) for sense 1.
__host__ __device__ __forceinline__ void flat_to_xy(int n, int corner, int sense, int row, int col, int& x, int& y) {
    const int u = sense ? row : col, v = sense ? col : row;
    switch (corner) {
        case 0: x = u; y = v; break;
        case 1: x = n - 1 - v; y = u; break;
        case 2: x = n - 1 - u; y = n - 1 - v; break;
        default: x = v; y = n - 1 - u; break;
    }
}
__host__ __device__ __forceinline__ void xy_to_flat(int n, int corner, int sense, int x, int y, int& row, int& col) {
    int u, v;
    switch (corner) {
        case 0: u = x; v = y; break;
        case 1: u = y; v = n - 1 - x; break;
        case 2: u = n - 1 - x; v = n - 1 - y; break;
        default: u = n - 1 - y; v = x; break;
    }
    col = sense ? v : u;
    row = sense ? u : v;
}
__host__ __device__ __forceinline__ unsigned long long spread_bits(unsigned v) {  // bit b -> bit 2 b
    unsigned long long r = v;
    r = (r | (r << 16)) & 0x0000ffff0000ffffULL;
    r = (r | (r << 8)) & 0x00ff00ff00ff00ffULL;
    r = (r | (r << 4)) & 0x0f0f0f0f0f0f0f0fULL;
    r = (r | (r << 2)) & 0x3333333333333333ULL;
    r = (r | (r << 1)) & 0x5555555555555555ULL;
    return r;
}
// non-RING layouts: index <-> (x, y, f)
__host__ __device__ __forceinline__ void index_to_xyf(int n, int layout, long long ip, int& x, int& y, int& f) {
    const long long n2 = (long long)n * n;
    f = (int)(ip / n2);
    const long long r = ip - (long long)f * n2;
    if (layout == 1) {
        x = (int)compact_bits((unsigned long long)r);
        y = (int)compact_bits((unsigned long long)r >> 1);
    } else {
        flat_to_xy(n, (layout - 2) >> 1, (layout - 2) & 1, (int)(r / n), (int)(r % n), x, y);
    }
}
__host__ __device__ __forceinline__ long long xyf_to_index(int n, int layout, int x, int y, int f) {
    if (layout == 0) return xyf_to_ring(n, x, y, f);
    const long long n2 = (long long)n * n;
    if (layout == 1) return f * n2 + (long long)(spread_bits((unsigned)x) | (spread_bits((unsigned)y) << 1));
    int row, col;
    xy_to_flat(n, (layout - 2) >> 1, (layout - 2) & 1, x, y, row, col);
    return f * n2 + (long long)row * n + col;
}

// `walk` is a non-RING layout: thread i handles the pixel with index i in that layout (coalesced on that side);
// GATHER: out[i] = in[other(i)] (walk = destination);  otherwise out[other(i)] = in[i] (walk = source).
template <typename W, bool GATHER>
__global__ void __launch_bounds__(256) layout_kernel(int nside, long long npix, int walk, int other, const W* __restrict__ in,
                                                     W* __restrict__ out) {
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (i >= npix) return;
    int x, y, f;
    index_to_xyf(nside, walk, i, x, y, f);
    const long long j = xyf_to_index(nside, other, x, y, f);
    const size_t b = (size_t)blockIdx.y * (size_t)npix;
    if (GATHER) out[b + i] = in[b + j];
    else out[b + j] = in[b + i];
}

long long layout_index(int nside, int src_layout, int dst_layout, long long ip_src) {
    // only used by the host helper: RING as a source has no closed form here -> search is the caller's business
    int x, y, f;
    index_to_xyf(nside, src_layout, ip_src, x, y, f);
    return xyf_to_index(nside, dst_layout, x, y, f);
}

cudaError_t launch_layout(int nside, int batch, cuhpx_dtype_t dt, int src, int dst, const void* in, void* out, cudaStream_t st) {
    if (src == dst) {
        const size_t bytes = (size_t)batch * 12 * nside * nside * (dt == CUHPX_F64 ? 8 : 4);
        return cudaMemcpyAsync(out, in, bytes, cudaMemcpyDeviceToDevice, st);
    }
    if ((src == 0 && dst == 1) || (src == 1 && dst == 0)) return launch_reorder(nside, batch, dt, dst == 0, in, out, st);
    const long long npix = 12LL * nside * nside;
    const dim3 grid((unsigned)((npix + 255) / 256), (unsigned)batch);
    const bool gather = src == 0 || dst != 0;  // walk the destination unless the destination is RING
    const int walk = gather ? dst : src, other = gather ? src : dst;
    if (dt == CUHPX_F64) {
        if (gather) layout_kernel<uint64_t, true><<<grid, 256, 0, st>>>(nside, npix, walk, other, (const uint64_t*)in, (uint64_t*)out);
        else layout_kernel<uint64_t, false><<<grid, 256, 0, st>>>(nside, npix, walk, other, (const uint64_t*)in, (uint64_t*)out);
    } else {
        if (gather) layout_kernel<uint32_t, true><<<grid, 256, 0, st>>>(nside, npix, walk, other, (const uint32_t*)in, (uint32_t*)out);
        else layout_kernel<uint32_t, false><<<grid, 256, 0, st>>>(nside, npix, walk, other, (const uint32_t*)in, (uint32_t*)out);
    }
    return cudaGetLastError();
}

// ------------------------------------------------------------------ spectral resampling
// "upsampling and downsampling of HEALPix data by truncating or extending spherical harmonic coefficients before
// applying the iSHT": out(l, m) = in(l, m) where the input has that coefficient, else 0.  W = one complex value.
template <typename W>
__global__ void __launch_bounds__(256) alm_resize_kernel(int lmax_in, int mmax_in, int lmax_out, long long nalm_in,
                                                         long long nalm_out, const W* __restrict__ in, W* __restrict__ out) {
    const int m = blockIdx.x, b = blockIdx.y;
    const long long base_out = (long long)m * (2LL * lmax_out + 1 - m) / 2;  // index of (l = 0, m), m-major packed
    const long long base_in = (long long)m * (2LL * lmax_in + 1 - m) / 2;
    W zero;
    memset(&zero, 0, sizeof(W));
    for (int l = m + threadIdx.x; l <= lmax_out; l += blockDim.x) {
        const bool have = m <= mmax_in && l <= lmax_in;
        out[(size_t)b * nalm_out + base_out + l] = have ? in[(size_t)b * nalm_in + base_in + l] : zero;
    }
}

cudaError_t launch_alm_resize(int lmax_in, int mmax_in, int lmax_out, int mmax_out, int batch, cuhpx_dtype_t dt,
                              const void* in, void* out, cudaStream_t st) {
    const long long nin = (long long)(mmax_in + 1) * (lmax_in + 1) - (long long)mmax_in * (mmax_in + 1) / 2;
    const long long nout = (long long)(mmax_out + 1) * (lmax_out + 1) - (long long)mmax_out * (mmax_out + 1) / 2;
    dim3 grid((unsigned)(mmax_out + 1), (unsigned)batch);
    if (dt == CUHPX_F64) alm_resize_kernel<double2><<<grid, 256, 0, st>>>(lmax_in, mmax_in, lmax_out, nin, nout, (const double2*)in, (double2*)out);
    else alm_resize_kernel<float2><<<grid, 256, 0, st>>>(lmax_in, mmax_in, lmax_out, nin, nout, (const float2*)in, (float2*)out);
    return cudaGetLastError();
}

}  // namespace cuhpx

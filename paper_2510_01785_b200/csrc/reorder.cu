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
__host__ __device__ __forceinline__ unsigned long long spread_bits(unsigned v) {
    unsigned long long w = v;
    w = (w | (w << 16)) & 0x0000ffff0000ffffull;
    w = (w | (w << 8)) & 0x00ff00ff00ff00ffull;
    w = (w | (w << 4)) & 0x0f0f0f0f0f0f0f0full;
    w = (w | (w << 2)) & 0x3333333333333333ull;
    w = (w | (w << 1)) & 0x5555555555555555ull;
    return w;
}

long long nest_to_ring_index(int nside, long long ipnest) {
    const long long ns2 = (long long)nside * nside;
    const int f = (int)(ipnest / ns2);
    const unsigned long long r = (unsigned long long)(ipnest % ns2);
    return xyf_to_ring(nside, (int)compact_bits(r), (int)compact_bits(r >> 1), f);
}

constexpr int RT_THREADS = 256;

// T = tile edge (power of two, <= 64, <= nside).  grid.x = 12 (nside / T)^2 tiles, grid.y = batch.
template <typename W, int T, bool TO_RING>
__global__ void __launch_bounds__(RT_THREADS) reorder_kernel(int nside, long long npix, const W* __restrict__ in, W* __restrict__ out) {
    __shared__ W tile[T * T];
    const int tiles_per_face = (nside / T) * (nside / T);
    const int f = blockIdx.x / tiles_per_face;
    const unsigned tmorton = blockIdx.x % tiles_per_face;  // tiles of a face in Z-order, like the pixels
    const int x0 = (int)compact_bits(tmorton) * T, y0 = (int)compact_bits(tmorton >> 1) * T;
    const long long nest0 = (long long)f * nside * nside + (long long)tmorton * (T * T);
    const W* src = in + (size_t)blockIdx.y * npix;
    W* dst = out + (size_t)blockIdx.y * npix;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    if (TO_RING) {
        for (int e = tid; e < T * T; e += RT_THREADS) {
            const int xl = (int)compact_bits((unsigned)e), yl = (int)compact_bits((unsigned)e >> 1);
            tile[yl * T + xl] = src[nest0 + e];
        }
        __syncthreads();
    }
    // anti-diagonals s = xl + yl of the block: consecutive xl are consecutive pixels of one ring
    for (int s = warp; s < 2 * T - 1; s += RT_THREADS / 32) {
        const int xmin = s < T ? 0 : s - T + 1, len = s < T ? s + 1 : 2 * T - 1 - s;
        for (int k = lane; k < len; k += 32) {
            const int xl = xmin + k, yl = s - xl;
            const long long ir = xyf_to_ring(nside, x0 + xl, y0 + yl, f);
            if (TO_RING) dst[ir] = tile[yl * T + xl];
            else tile[yl * T + xl] = src[ir];
        }
    }
    if (!TO_RING) {
        __syncthreads();
        for (int e = tid; e < T * T; e += RT_THREADS) {
            const int xl = (int)compact_bits((unsigned)e), yl = (int)compact_bits((unsigned)e >> 1);
            dst[nest0 + e] = tile[yl * T + xl];
        }
    }
}

template <typename W, int T>
static cudaError_t run_reorder_t(int nside, int batch, int to_ring, const void* in, void* out, cudaStream_t st) {
    const long long npix = 12LL * nside * nside;
    dim3 grid((unsigned)(12 * (nside / T) * (nside / T)), (unsigned)batch);
    if (to_ring) reorder_kernel<W, T, true><<<grid, RT_THREADS, 0, st>>>(nside, npix, (const W*)in, (W*)out);
    else reorder_kernel<W, T, false><<<grid, RT_THREADS, 0, st>>>(nside, npix, (const W*)in, (W*)out);
    return cudaGetLastError();
}

template <typename W>
static cudaError_t run_reorder(int nside, int batch, int to_ring, const void* in, void* out, cudaStream_t st) {
    if (nside >= 64) return run_reorder_t<W, 64>(nside, batch, to_ring, in, out, st);
    if (nside >= 16) return run_reorder_t<W, 16>(nside, batch, to_ring, in, out, st);
    if (nside >= 4) return run_reorder_t<W, 4>(nside, batch, to_ring, in, out, st);
    return run_reorder_t<W, 1>(nside, batch, to_ring, in, out, st);
}

cudaError_t launch_reorder(int nside, int batch, cuhpx_dtype_t dt, int to_ring, const void* in, void* out, cudaStream_t st) {
    return dt == CUHPX_F64 ? run_reorder<uint64_t>(nside, batch, to_ring, in, out, st)
                           : run_reorder<uint32_t>(nside, batch, to_ring, in, out, st);
}

}  // namespace cuhpx

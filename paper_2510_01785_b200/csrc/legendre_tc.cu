// Legendre stage on the Blackwell tensor path (tcgen05 + tensor memory) for batched fp32 transforms
// (north_star: "tensor cores ... where the Legendre stage really is a dense contraction, meaning batched channels
// with lambda tiles amortised"; SURVEY 8(d) "Batched Legendre"; Eq. 14, Eq. 24, Eq. 26).
//
// Synthesis (row s1), per order m:   G[j][c] = sum_l Lambda[l][j] (s_l a[l][c]),   j = ring pair, c = (channel, re/im)
//   M = 128 ring pairs (one per thread = one tensor-memory lane), K = degrees l of one parity, N = columns c.
//   Every thread walks the fp64 recurrence of its ring pairs and writes lambda -- split in two TF32 terms,
//   lambda = hi + lo -- straight into tensor memory as the A operand (tcgen05.st: lane = ring, column = degree):
//   lambda never touches shared memory.  The B operand (s_l a_lm, also split hi + lo, K-major [hi | lo] columns) is
//   laid out once per call by a small pre-pass kernel (synthesis_images_kernel) as ready-to-use "images" in the
//   workspace -- per (channel group, order m, stage of 32 degrees): the 32 recurrence coefficients alpha and four
//   K = 8 tiles [parity][K block] -- which the main kernel fetches with one bulk asynchronous copy (TMA, mbarrier
//   complete_tx) per stage, three in flight.  Per 8 degrees of one parity two instructions
//       D(128 x 4 NB) += A_hi (TMEM) x [a_hi | a_lo],      D(128 x 2 NB) += A_lo (TMEM) x [a_hi]
//   give hi hi + hi lo + lo hi (the dropped lo lo term is 2^-22 relative); the accumulators E (even l - m) and
//   O (odd) live in tensor memory and come back once, at the end: G(N) = E + O, G(S) = E - O.
//   CTA = 4 producer warps (one 128-ring tile) + one warp that requests the images and issues the tcgen05.mma of a
//   stage when the producers have parked it (mbarrier `ready`), committing to the mbarrier (`bar`) the producers wait
//   on before they overwrite the lambda buffer; the next stage is generated into registers meanwhile.  128 columns of
//   tensor memory per CTA at NB = 8: four CTAs per SM.
//   Variants measured and dropped (cfg4, 2.37 ms as built): two tiles per CTA 2.58 ms; lambda double-buffered by
//   half-stages of 16 degrees 2.59 ms; two ring pairs per producer thread 2.66 ms; two producer threads per ring pair
//   (one per parity, duplicated recurrence) 3.61 ms.  With an empty pipeline (no recurrence, no MMA) the kernel takes
//   0.86 ms: 0.48 ms per-CTA fixed cost (seeds, first image, the strided 8-byte epilogue stores) + 0.38 ms of per-stage
//   synchronisation.
#include <cuda_runtime.h>
#include <math.h>
#include <stdlib.h>

#include "cuhpx_internal.h"
#include "legendre_common.cuh"
#include "tc_common.cuh"

namespace cuhpx {

namespace {

constexpr int TC_TILE = 128;    // ring pairs per tile: one per thread of a 4-warp group = one tensor-memory lane each
constexpr int TC_STAGE = 32;    // degrees per stage: 16 even + 16 odd (l - m) = two K = 8 instruction pairs per parity

__host__ __device__ constexpr int pow2_at_least(int v) {
    int p = 32;
    while (p < v) p *= 2;
    return p;
}

// tensor-memory columns: accumulators [tile][parity][4 NB], then the lambda buffer [tile][parity][hi, lo][16]
template <int NB, int TILES> struct SynthTmem {
    static constexpr int N1 = 4 * NB, N2 = 2 * NB;
    static constexpr int D_COLS = TILES * 2 * N1;
    static constexpr int A_COLS = TILES * 64;
    static constexpr int COLS = pow2_at_least(D_COLS + A_COLS);
    static_assert(COLS <= 512, "tensor memory");
    static_assert(N1 <= 256 && N2 % 16 == 0, "instruction shape");
    __host__ __device__ static constexpr int d_col(int tile, int par) { return (tile * 2 + par) * N1; }
    __host__ __device__ static constexpr int a_col(int tile, int par, int hl) { return D_COLS + (tile * 2 + par) * 32 + hl * 16; }
};

// shared-memory B tile of one (buffer, parity, K block): K = 8 degrees x N1 columns, tf32, K-major, no swizzle:
// element (n, k) at float offset (n % 8) * 4 + (n / 8) * 64 + (k % 4) + (k / 4) * 32   (LBO = 128 B, SBO = 256 B)
__device__ __forceinline__ int btile_off(int n, int k) { return (n & 7) * 4 + (n >> 3) * 64 + (k & 3) + (k >> 2) * 32; }

// Operand image of one (channel group, order m, stage of 32 degrees), built per call by synthesis_images_kernel and
// fetched by the main kernel with one bulk copy (TMA):  [alpha of the 32 steps: 32 doubles][B tiles [parity][K block]]
template <int NB> struct SynthImage {
    static constexpr int N1 = 4 * NB;
    static constexpr int BTILE = 8 * N1;  // floats per tile
    static constexpr int BYTES = 256 + 4 * BTILE * 4;
    __host__ __device__ static constexpr int tile_off(int par, int kb) { return 256 + (par * 2 + kb) * BTILE * 4; }  // bytes
};

}  // namespace

int legendre_tc_group(cuhpx_dtype_t dt, int batch) { return (dt == CUHPX_F32 && batch >= 8) ? (batch >= 16 ? 16 : 8) : 0; }
size_t legendre_tc_image_bytes(int nb) { return nb == 16 ? SynthImage<16>::BYTES : SynthImage<8>::BYTES; }

// One CTA per (order m, channel group): s_l a_lm (times 1/c_m for the adjoint), split in hi + lo TF32 terms, laid out as
// the K-major B operand [hi (2 NB columns) | lo (2 NB)] of every stage, plus the recurrence coefficients alpha.
template <int NB>
__global__ void __launch_bounds__(256) synthesis_images_kernel(LegArgs a) {
    using IM = SynthImage<NB>;
    constexpr int N2 = 2 * NB, NT = 256;
    constexpr int SRC = (TC_STAGE * NB + NT - 1) / NT;
    const DevPlan& P = a.p;
    if (!ws_ok(P)) return;
    const int m = blockIdx.x, g = blockIdx.y, ch0 = g * NB;
    const int tid = threadIdx.x, lane = tid & 31;
    __shared__ __align__(16) unsigned char img[IM::BYTES];
    const float inscale = (a.adjoint && m > 0) ? 0.5f : 1.f;
    const long long abase = (long long)m * (2LL * P.lmax + 1 - m) / 2;
    const float* alm = reinterpret_cast<const float*>(a.in);
    const int nl = P.lmax - m + 1;
    const int nstage = (nl + TC_STAGE - 1) / TC_STAGE;
    const long long total = P.tc_prefix[P.mmax + 1];
    unsigned char* out = reinterpret_cast<unsigned char*>(P.tc_images) + ((size_t)g * total + P.tc_prefix[m]) * IM::BYTES;
    for (int s = 0; s < nstage; ++s) {
        const int l0 = s * TC_STAGE;
        // a warp covers 8 consecutive degrees of 4 channels (64-byte runs in global memory, all shared-memory banks)
#pragma unroll
        for (int q = 0; q < SRC; ++q) {
            const int e = tid + q * NT, wq = e >> 5;
            const int i = 8 * (wq & 3) + 2 * ((lane >> 2) & 3) + (lane >> 4);
            const int c = 4 * (wq >> 2) + (lane & 3);
            if (c < NB) {
                const int k = l0 + i, ch = ch0 + c;
                const bool ok = k < nl && ch < P.batch;
                const float2 v = ok ? *reinterpret_cast<const float2*>(&alm[((size_t)ch * P.nalm + abase + m + k) * 2]) : make_float2(0.f, 0.f);
                const float sl = ok ? (float)((double)inscale * P.coef_scale[abase + m + k]) : 0.f;
                float vr = sl * v.x, vi = sl * v.y;
                if (m == 0) vi = 0.f;  // Im a_l0 is ignored
                uint32_t hr, lr, hi, li;
                tc::split_tf32(vr, hr, lr);
                tc::split_tf32(vi, hi, li);
                uint32_t* tl = reinterpret_cast<uint32_t*>(img + IM::tile_off(i & 1, i >> 4));
                const int kk = (i >> 1) & 7;
                tl[btile_off(2 * c, kk)] = hr;
                tl[btile_off(2 * c + 1, kk)] = hi;
                tl[btile_off(N2 + 2 * c, kk)] = lr;
                tl[btile_off(N2 + 2 * c + 1, kk)] = li;
            }
        }
        if (tid < TC_STAGE) reinterpret_cast<double*>(img)[tid] = (l0 + 1 + tid < nl) ? P.coef_alpha[abase + m + l0 + 1 + tid] : 0.0;
        __syncthreads();
        float4* dst = reinterpret_cast<float4*>(out + (size_t)s * IM::BYTES);
        for (int e = tid; e < IM::BYTES / 16; e += NT) dst[e] = reinterpret_cast<const float4*>(img)[e];
        __syncthreads();
    }
}

template <int NB, int TILES>
__global__ void __launch_bounds__(TC_TILE * TILES + 32) legendre_synthesis_tc_kernel(LegArgs a) {
    using TM = SynthTmem<NB, TILES>;
    using IM = SynthImage<NB>;
    constexpr int NP = TC_TILE * TILES;  // producer threads (ring pairs); one more warp issues the tensor-core work
    constexpr int N1 = TM::N1, N2 = TM::N2;
    constexpr int NBUF = 3;  // stage images in flight
    const DevPlan& P = a.p;
    if (!ws_ok(P)) return;
    const int m = blockIdx.y;
    const int chunk = blockIdx.x;
    const int ch0 = blockIdx.z * NB;
    const int tid = threadIdx.x, warp = tid >> 5;
    const int jbase = P.jmin[m] + chunk * NP;
    if (jbase >= P.npairs) return;

    __shared__ __align__(128) unsigned char img[NBUF][IM::BYTES];
    __shared__ __align__(8) uint64_t full[NBUF];  // image landed (TMA complete_tx)
    __shared__ __align__(8) uint64_t ready;       // every producer warp has parked its lambda of the stage in tensor memory
    __shared__ __align__(8) uint64_t bar;         // tensor-core instructions of a stage completed
    __shared__ uint32_t tmem_slot;

    const int nl = P.lmax - m + 1;
    const int nstage = (nl + TC_STAGE - 1) / TC_STAGE;
    const bool issuer = warp == NP / 32;
    if (issuer) tc::tmem_alloc(&tmem_slot, TM::COLS);
    if (tid == NP) {
        tc::mbar_init(&bar, 1);
        tc::mbar_init(&ready, NP / 32);
#pragma unroll
        for (int b = 0; b < NBUF; ++b) tc::mbar_init(&full[b], 1);
        tc::fence_mbar_init();
    }
    tc::fence_before_sync();
    __syncthreads();
    tc::fence_after_sync();
    const uint32_t tbase = tmem_slot;

    if (issuer) {
        // ================= issuing warp: image requests (TMA) and tcgen05.mma for every stage
        if (tid == NP) {
            const unsigned char* images = reinterpret_cast<const unsigned char*>(P.tc_images) +
                                          ((size_t)blockIdx.z * P.tc_prefix[P.mmax + 1] + P.tc_prefix[m]) * IM::BYTES;
            auto request = [&](int s) {  // image of stage s -> buffer s % NBUF
                tc::mbar_arrive_expect_tx(&full[s % NBUF], IM::BYTES);
                tc::bulk_g2s(img[s % NBUF], images + (size_t)s * IM::BYTES, IM::BYTES, &full[s % NBUF]);
            };
            for (int s = 0; s < NBUF && s < nstage; ++s) request(s);
            constexpr uint32_t id1 = tc::idesc_tf32(128, N1), id2 = tc::idesc_tf32(128, N2);
            for (int s = 0; s < nstage; ++s) {
                const int buf = s % NBUF;
                tc::mbar_wait(&ready, (uint32_t)(s & 1));
                tc::fence_after_sync();
                // the producers awaited the instructions of stage s - 1 before they parked stage s: image (s - 1) % NBUF is free
                if (s >= 1 && s + 2 < nstage) request(s + 2);
                tc::mbar_wait(&full[buf], (uint32_t)((s / NBUF) & 1));
                // consecutive instructions go to different accumulators (E / O, tiles): back-to-back instructions on one
                // accumulator wait for each other
#pragma unroll
                for (int kb = 0; kb < 2; ++kb) {
                    const uint64_t bde = tc::smem_desc(tc::smem_u32(img[buf] + IM::tile_off(0, kb)), 128, 256);
                    const uint64_t bdo = tc::smem_desc(tc::smem_u32(img[buf] + IM::tile_off(1, kb)), 128, 256);
#pragma unroll
                    for (int hl = 0; hl < 2; ++hl) {
#pragma unroll
                        for (int t = 0; t < TILES; ++t) {
                            const uint32_t acc = (s > 0 || kb > 0 || hl > 0) ? 1u : 0u;
                            tc::mma_tf32_ts(tbase + TM::d_col(t, 0), tbase + TM::a_col(t, 0, hl) + kb * 8, bde, hl ? id2 : id1, acc);
                            tc::mma_tf32_ts(tbase + TM::d_col(t, 1), tbase + TM::a_col(t, 1, hl) + kb * 8, bdo, hl ? id2 : id1, acc);
                        }
                    }
                }
                tc::umma_commit(&bar);
            }
        }
        __syncwarp();
    } else {
        // ================= producer warps: one ring pair per thread
        const int tile = warp >> 2;                                        // the 4-warp group's ring tile
        const uint32_t lane_field = (uint32_t)((warp & 3) * 32) << 16;     // a warp reaches the lane quadrant warp % 4
        double cur = 0.0, prev = 0.0, cx = 0.0;
        int sc = -1;
        const int j = jbase + tid;
        if (j < P.npairs) {
            cx = 1.0 - P.y[j];  // cos(theta): fp32 output (R8)
            lambda_seed<float>(m, P.pref_hi[m], P.pref_lo[m], P.ls_hi[j], P.ls_lo[j], cur, sc);
        }
        bool all_on = false;  // warp-uniform: every ring pair of this warp is significant (no more checks, no selects)
        for (int s = 0; s < nstage; ++s) {
            const int buf = s % NBUF;
            tc::mbar_wait(&full[buf], (uint32_t)((s / NBUF) & 1));
            const double* sA = reinterpret_cast<const double*>(img[buf]);
            // ---- 32 degrees into registers (the previous stage's instructions still read the tensor-memory buffer)
            uint32_t eh[16], el[16], oh[16], ol[16];
            if (all_on) {
#pragma unroll
                for (int p = 0; p < 16; ++p) {
                    tc::split_tf32((float)cur, eh[p], el[p]);
                    double nx = fma(sA[2 * p] * cx, cur, -prev);
                    prev = cur;
                    cur = nx;
                    tc::split_tf32((float)cur, oh[p], ol[p]);
                    nx = fma(sA[2 * p + 1] * cx, cur, -prev);
                    prev = cur;
                    cur = nx;
                }
            } else {
#pragma unroll
                for (int h = 0; h < 4; ++h) {
                    if (sc < 0 && fabs(cur) > pow2c(ScaleCfg<float>::THR)) {
                        cur *= pow2c(-ScaleCfg<float>::K);
                        prev *= pow2c(-ScaleCfg<float>::K);
                        ++sc;
                    }
                    const bool on = sc == 0;
#pragma unroll
                    for (int p = 0; p < 4; ++p) {
                        const int i = h * 8 + 2 * p;
                        float v = on ? (float)cur : 0.f;
                        tc::split_tf32(v, eh[h * 4 + p], el[h * 4 + p]);
                        double nx = fma(sA[i] * cx, cur, -prev);
                        prev = cur;
                        cur = nx;
                        v = on ? (float)cur : 0.f;
                        tc::split_tf32(v, oh[h * 4 + p], ol[h * 4 + p]);
                        nx = fma(sA[i + 1] * cx, cur, -prev);
                        prev = cur;
                        cur = nx;
                    }
                }
                all_on = __all_sync(0xffffffffu, sc == 0);
            }
            if (s >= 1) {  // the instructions of stage s - 1 have completed: the lambda buffer is free
                tc::mbar_wait(&bar, (uint32_t)((s - 1) & 1));
                tc::fence_after_sync();
            }
            tc::tmem_st16(tbase + lane_field + TM::a_col(tile, 0, 0), eh);
            tc::tmem_st16(tbase + lane_field + TM::a_col(tile, 0, 1), el);
            tc::tmem_st16(tbase + lane_field + TM::a_col(tile, 1, 0), oh);
            tc::tmem_st16(tbase + lane_field + TM::a_col(tile, 1, 1), ol);
            tc::tmem_wait_st();
            tc::fence_before_sync();
            __syncwarp();
            if ((tid & 31) == 0) tc::mbar_arrive(&ready);
        }
        // ---- every instruction has completed once the last commit has arrived (each earlier one was awaited above)
        tc::mbar_wait(&bar, (uint32_t)((nstage - 1) & 1));
        tc::fence_after_sync();
    float2* spectra = reinterpret_cast<float2*>(P.spectra);
    {
        const int rn = j, rs = P.nrings - 1 - j;
        const bool live = j < P.npairs && sc == 0;
#pragma unroll
        for (int c0 = 0; c0 < N2; c0 += 16) {  // 8 channels at a time
            uint32_t qeh[16], qel[16], qoh[16], qol[16];
            tc::tmem_ld16(tbase + lane_field + TM::d_col(tile, 0) + c0, qeh);
            tc::tmem_ld16(tbase + lane_field + TM::d_col(tile, 0) + N2 + c0, qel);
            tc::tmem_ld16(tbase + lane_field + TM::d_col(tile, 1) + c0, qoh);
            tc::tmem_ld16(tbase + lane_field + TM::d_col(tile, 1) + N2 + c0, qol);
            tc::tmem_wait_ld();
            if (j < P.npairs) {
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    const int ch = ch0 + (c0 >> 1) + c;
                    if (ch >= P.batch) continue;
                    const float er = __uint_as_float(qeh[2 * c]) + __uint_as_float(qel[2 * c]);
                    const float ei = __uint_as_float(qeh[2 * c + 1]) + __uint_as_float(qel[2 * c + 1]);
                    const float orr = __uint_as_float(qoh[2 * c]) + __uint_as_float(qol[2 * c]);
                    const float oi = __uint_as_float(qoh[2 * c + 1]) + __uint_as_float(qol[2 * c + 1]);
                    float2 gn = make_float2(0.f, 0.f), gs = gn;
                    if (live) {
                        gn = make_float2(er + orr, ei + oi);
                        gs = make_float2(er - orr, ei - oi);
                    }
                    spectra[((size_t)ch * P.nrings + rn) * P.mstride + m] = gn;
                    if (rs != rn) spectra[((size_t)ch * P.nrings + rs) * P.mstride + m] = gs;
                }
            }
        }
    }
    }  // producer warps
    tc::fence_before_sync();
    __syncthreads();
    if (issuer) tc::tmem_dealloc(tbase, TM::COLS);
}

// ------------------------------------------------------------------ launchers
bool legendre_tc_enabled() {
    // CUHPX_LEGENDRE_TC=0 selects the CUDA-core kernels of legendre.cu instead (A/B measurements, profiles/r2_*.md)
    static const bool on = [] {
        const char* e = getenv("CUHPX_LEGENDRE_TC");
        return !(e && e[0] == '0');
    }();
    return on;
}

template <int NB, int TILES>
static cudaError_t run_synthesis_tc(const DevPlan& P, const void* d_alm, int adjoint, cudaStream_t st) {
    LegArgs a;
    a.p = P;
    a.in = d_alm;
    a.out = nullptr;
    a.adjoint = adjoint;
    a.to_partial = 0;
    const int chunk = TC_TILE * TILES;
    dim3 grid((P.npairs + chunk - 1) / chunk, P.mmax + 1, (P.batch + NB - 1) / NB);
    synthesis_images_kernel<NB><<<dim3(P.mmax + 1, (P.batch + NB - 1) / NB), 256, 0, st>>>(a);
    legendre_synthesis_tc_kernel<NB, TILES><<<grid, TC_TILE * TILES + 32, 0, st>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_legendre_synthesis_tc(const HostPlan& hp, const DevPlan& P, const void* d_alm, int adjoint, cudaStream_t st) {
    if (P.tc_nb == 0 || !P.tc_images || !legendre_tc_enabled()) return cudaErrorNotSupported;
    // one 128-ring tile per CTA (128 tensor-memory columns at NB = 8: four CTAs per SM in different phases keep the
    // FP64 pipe and the tensor pipe busier than two CTAs of two tiles: 2.37 vs 2.58 ms at BASELINE configs[3])
    if (P.tc_nb == 16) return run_synthesis_tc<16, 1>(P, d_alm, adjoint, st);
    return run_synthesis_tc<8, 1>(P, d_alm, adjoint, st);
}

}  // namespace cuhpx

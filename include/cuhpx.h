/*
 * cuhpx.h -- C ABI of the B200-native HEALPix spherical harmonic transform (cuHPX hot path,
 * arXiv 2510.01785; citations "P:n" are line n of the paper text, SURVEY.md section 8 is the scope table).
 *
 * The four operators on RING-ordered HEALPix maps, as real-linear maps between
 *   map  : [batch][npix]  real (dtype),            npix = 12 nside^2
 *   alm  : [batch][nalm]  complex interleaved (re,im) of dtype, m-major packed:
 *          index(l, m) = m (2 lmax + 1 - m) / 2 + l,   0 <= m <= mmax <= lmax,  m <= l <= lmax (inclusive)
 *
 *   cuhpx_alm2map          S   : p_xy = sum_m sum_l a_lm lambda_lm(theta_y) exp(i m (phi0_y + 2 pi x / N_y))   Eq. 24
 *                                (m < 0 terms implied by reality of the map; Im a_l0 is ignored)
 *   cuhpx_map2alm          A   : a_lm = sum_y sum_x p_xy w_y lambda_lm(theta_y) exp(-i m (phi0_y + 2 pi x / N_y)) Eq. 26
 *                                (a = Y^dagger W p, Eq. 27; output Im a_l0 is exactly 0)
 *   cuhpx_alm2map_adjoint  S^T : "adjoint iSHT = Y^dagger"  P:287;  (S^T g)_lm = c_m sum_p g_p lambda_lm exp(-i m phi_p)
 *   cuhpx_map2alm_adjoint  A^T : "adjoint SHT = W Y"        P:288;  (A^T b)_p = w_p [sum_l Re(b_l0) lambda_l0
 *                                                                        + sum_{m>=1} sum_l Re(b_lm lambda_lm exp(i m phi_p))]
 *   with c_0 = 1, c_m = 2 (m >= 1).  The transposes are taken w.r.t. <f,g> = sum_p f_p g_p and
 *   <a,b> = sum_{l, m>=0} (Re a Re b + Im a Im b): the inner product autograd uses for the stored tensor, so
 *   these are the analytic gradients of S and A.  A = D^-1 S^T W with D = diag(c_m).
 *
 * lambda_lm is the normalised associated Legendre function of Eq. 15 (Condon-Shortley phase included),
 * generated on the fly by the three-term recurrence of Eq. 16; ring geometry follows Gorski et al.
 * (ref [1] P:416): rings i = 1..4 nside - 1 north to south, polar caps N_i = 4 i, belt N_i = 4 nside.
 *
 * Conventions
 *   - Every data pointer is a DEVICE pointer owned by the caller, 16-byte aligned.  The library allocates no
 *     device memory: scratch and constant tables live in the caller's workspace (cuhpx_workspace_bytes).
 *   - The library keeps no per-workspace state and no call has to be paired with a free: a workspace is plain
 *     device memory whose first 256 bytes are a header (magic, parameter key) written by cuhpx_workspace_init.  It
 *     may be copied or moved (tables are addressed relative to the pointer passed to each call) and is simply
 *     freed by its owner.  What the host needs per call (ring classes, cut-offs, launch shapes, table offsets) is a
 *     pure function of (nside, lmax, mmax, batch, dtype), memoised inside the library.  Every kernel checks the
 *     header first: a call on memory that was not initialised for the same five parameters does nothing except
 *     marking the header (cuhpx_workspace_check reports it); it never follows a pointer from a foreign table.
 *   - Inputs are const, outputs are fully overwritten (never accumulated); input, output and workspace ranges must
 *     not overlap (checked on the host, CUHPX_EINVAL).
 *   - All work is enqueued on `stream`; the transform calls never synchronise with the host and can be captured
 *     in a CUDA graph (tests/test_gpu_parity.py::test_cuda_graph_capture_replay).  Part of the FFT stage runs on a
 *     library stream forked from and joined to `stream` with events (created once per device, never per
 *     workspace).  cuhpx_workspace_init enqueues table-building kernels and host->device copies on `stream` and
 *     returns after they have completed.  A workspace serves one transform at a time (calls sharing one workspace
 *     must be stream-ordered).
 *   - ring_weights: DEVICE pointer to 4 nside - 1 doubles (always fp64), rings north to south, the full
 *     quadrature weight w_y of Eq. 26 (i.e. including the 4 pi / Npix factor); NULL = equal weights
 *     4 pi / Npix (Eq. 1).
 *   - Return value: a cuhpx_status_t.  Argument errors are detected on the host before any launch.  Nothing is
 *     thrown across the ABI.  After CUHPX_ECUDA, cudaGetLastError() describes the launch failure.
 *   - batch <= 65535 (channels index a grid dimension).
 *   - There is no CPU fallback: on a machine without a CUDA device every compute call returns CUHPX_ECUDA.
 *   - Two environment switches for A/B measurements only.  CUHPX_LEGENDRE_TC=0 (read once per process) runs batched
 *     fp32 Legendre synthesis (batch >= 8) on the CUDA-core kernels instead of the tcgen05 / tensor-memory kernel.
 *     CUHPX_LATE_START=0 (read when a parameter set is first planned) leaves out the late-start tables of the fp64
 *     Legendre kernels (20 bytes per (m, ring pair) and direction of workspace, transforms with >= 2048 ring pairs):
 *     every order is then walked from l = m.  Results are bit-identical either way.
 */
#ifndef CUHPX_H_
#define CUHPX_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum { CUHPX_F32 = 0, CUHPX_F64 = 1 } cuhpx_dtype_t;

/* ring grids the two stages can run on (cuhpx_grid_* calls below; the calls without "grid" are HEALPix) */
typedef enum { CUHPX_GRID_HEALPIX = 0, CUHPX_GRID_GAUSS_LEGENDRE = 1, CUHPX_GRID_EQUIANGULAR = 2 } cuhpx_grid_t;

typedef enum {
    CUHPX_OK = 0,
    CUHPX_EINVAL = 1,       /* bad nside / lmax / mmax / batch / dtype, null or misaligned pointer */
    CUHPX_EWORKSPACE = 2,   /* workspace too small, not initialised, or initialised for other parameters */
    CUHPX_EUNSUPPORTED = 3, /* valid request this build cannot serve (e.g. ring too long for one SM's shared memory) */
    CUHPX_ECUDA = 4         /* CUDA runtime / launch error */
} cuhpx_status_t;

/* a cudaStream_t (CUstream_st*), declared here so the header needs no CUDA include */
typedef struct CUstream_st* cuhpx_stream_t;

/* ---- host-only helpers (no device work) */
size_t cuhpx_npix(int nside);                      /* 12 nside^2; 0 if nside is not a power of two >= 1 */
size_t cuhpx_nrings(int nside);                    /* 4 nside - 1 */
size_t cuhpx_alm_count(int lmax, int mmax);        /* (mmax+1)(lmax+1) - mmax(mmax+1)/2; 0 on bad arguments */
size_t cuhpx_alm_index(int lmax, int l, int m);    /* m (2 lmax + 1 - m)/2 + l */
const char* cuhpx_status_string(int status);
/* Ring table of Gorski et al. as the library uses it (ring = 1 .. 4 nside - 1): pixel count, RING index of the
 * first pixel, cos(theta), phi0 of the first pixel.  Returns CUHPX_EINVAL on bad arguments. */
int cuhpx_ring_info(int nside, int ring, long long* n_pix, long long* first_pix, double* cos_theta, double* phi0);

/* ---- workspace */
/* Bytes of device workspace needed for (nside, lmax, mmax, batch, dtype); 0 on invalid arguments. */
size_t cuhpx_workspace_bytes(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype);
/* Build the constant tables (ring geometry, recurrence seeds and coefficients, twiddles, chirp filters) and the
 * header inside d_workspace.  Once per workspace; again if any of the five parameters changes.  Returns after the
 * tables are complete (it synchronises `stream`); config.tables_first_call_s in bench.py is the time of this call. */
int cuhpx_workspace_init(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, void* d_workspace,
                         size_t workspace_bytes, cuhpx_stream_t stream);
/* Optional, SYNCHRONISING: read the header back and report whether d_workspace is initialised for these parameters
 * and no kernel has refused it since (CUHPX_OK / CUHPX_EWORKSPACE). */
int cuhpx_workspace_check(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, const void* d_workspace,
                          size_t workspace_bytes, cuhpx_stream_t stream);

/* ---- the four operators */
int cuhpx_map2alm(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, const void* d_map, void* d_alm,
                  const double* d_ring_weights, void* d_workspace, size_t workspace_bytes, cuhpx_stream_t stream);
int cuhpx_alm2map(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, const void* d_alm, void* d_map,
                  void* d_workspace, size_t workspace_bytes, cuhpx_stream_t stream);
int cuhpx_alm2map_adjoint(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, const void* d_gmap,
                          void* d_galm, void* d_workspace, size_t workspace_bytes, cuhpx_stream_t stream);
int cuhpx_map2alm_adjoint(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, const void* d_galm,
                          void* d_gmap, const double* d_ring_weights, void* d_workspace, size_t workspace_bytes,
                          cuhpx_stream_t stream);

/* ---- iterative refinement of the analysis (Eq. 4; the paper's "future work")
 *   a^(0) = A f;   r^(k+1) = f - S a^(k);   a^(k+1) = a^(k) + A r^(k+1),   k = 0 .. n_iter - 1
 * with A = cuhpx_map2alm (ring weights as given) and S = cuhpx_alm2map.  n_iter = 0 is cuhpx_map2alm.  Each
 * iteration costs one synthesis and one analysis.  d_scratch_map ([batch][npix] real) and d_scratch_alm
 * ([batch][nalm] complex) are caller-owned scratch buffers of the transform's dtype, overwritten; on return
 * d_scratch_map holds the last residual r^(n_iter) (undefined for n_iter = 0).  Same conventions and error codes as
 * the four operators; n_iter < 0 or a null scratch pointer with n_iter > 0 is CUHPX_EINVAL. */
int cuhpx_map2alm_iter(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, const void* d_map, void* d_alm,
                       const double* d_ring_weights, int n_iter, void* d_scratch_map, void* d_scratch_alm,
                       void* d_workspace, size_t workspace_bytes, cuhpx_stream_t stream);

/* ---- ring quadrature weights ("cuHPX adopts ring weights as the default"; the paper
 * takes the values from the HEALPix data distribution, which is not available here -- DESIGN.md reading R11).
 * Writes 4 nside - 1 doubles w_i (rings north to south, including the 4 pi / Npix factor, i.e. directly usable as
 * d_ring_weights of cuhpx_map2alm / cuhpx_map2alm_iter / cuhpx_map2alm_adjoint) such that the m = 0 quadrature of Eq. 26
 * is exact:  sum_i w_i N_i lambda_l0(theta_i) = sqrt(4 pi) delta_l0  for every l <= lmax_w  (so a_l0 of a zonal map
 * band-limited to lmax_w / 2 is recovered to rounding), choosing among all such weights the one closest to equal weights,
 * min sum_i N_i (w_i - 4 pi / Npix)^2; the result is north/south symmetric.  lmax_w <= 0 selects the default 3 nside;
 * lmax_w > 3 nside is CUHPX_EINVAL (the Gram matrix of the zonal harmonics on the rings degenerates beyond).
 * Solved on the device with the m = 0 Legendre stages of the transform itself (conjugate gradients, ~50 iterations);
 * d_workspace: caller-owned DEVICE scratch of cuhpx_ring_weights_workspace_bytes() bytes, overwritten.  SYNCHRONISES
 * `stream` (table building + one read-back of the final residual); returns CUHPX_EUNSUPPORTED if the constraints are
 * not met to 1e-11. */
size_t cuhpx_ring_weights_workspace_bytes(int nside, int lmax_w);
int cuhpx_ring_weights(int nside, int lmax_w, double* d_weights, void* d_workspace, size_t workspace_bytes,
                       cuhpx_stream_t stream);

/* ---- the same solver for callers that may not allocate device memory (graph-capture set-up, serving loops, harnesses
 * that forbid cudaMalloc): the scratch is a built-in device array of CUHPX_NOALLOC_SCRATCH_BYTES (8 MiB) that every GPU
 * loading the library holds until the process exits; the call (and everything below it) makes no cudaMalloc / cudaFree
 * / allocating library call.  Same arguments, result and error codes as cuhpx_ring_weights without the workspace; a
 * request with cuhpx_ring_weights_workspace_bytes(nside, lmax_w) > CUHPX_NOALLOC_SCRATCH_BYTES (nside >= 1024 at the
 * default lmax_w) returns CUHPX_EWORKSPACE before anything is launched.  All calls on one device SHARE the array: it is
 * cleared at the start of each call, and two calls whose GPU work overlaps in time (other streams, other host threads)
 * race -- serialise them.  SYNCHRONISES `stream` like cuhpx_ring_weights. */
#define CUHPX_NOALLOC_SCRATCH_BYTES (8u << 20)
int cuhpx_ring_weights_noalloc(int nside, int lmax_w, double* d_weights, cuhpx_stream_t stream);

/* ---- layout reordering NESTED <-> RING (paper section III-B, via (x, y, f) P:118-123)
 * NESTED: index = f nside^2 + Z-order (Morton) interleave of (x, y) inside base face f (x on the even bits), P:109;
 * RING: as everywhere else in this header.  d_in / d_out: [batch][npix] elements of `dtype` (moved as bits,
 * 4 or 8 bytes each), DEVICE pointers, 16-byte aligned, must not alias.  direction: CUHPX_NEST2RING reads NESTED and
 * writes RING, CUHPX_RING2NEST the reverse.  No workspace.  Errors as for the operators. */
typedef enum { CUHPX_NEST2RING = 0, CUHPX_RING2NEST = 1 } cuhpx_reorder_t;
int cuhpx_reorder(int nside, int batch, cuhpx_dtype_t dtype, int direction, const void* d_in, void* d_out,
                  cuhpx_stream_t stream);
/* The three layouts of P:108-110 through the (x, y, f) intermediate of P:118-123.  Layout codes:
 *   CUHPX_LAYOUT_RING = 0, CUHPX_LAYOUT_NESTED = 1, CUHPX_LAYOUT_FLAT(corner, sense) = 2 + 2 corner + sense:
 * "flat" (Fig. 3C: "indexing requires both an orientation (clockwise or counterclockwise) and a reference point")
 * stores every base face as a row-major nside x nside image, index = f nside^2 + row nside + col, ready for 2-D
 * convolution kernels; the image origin is the face's corner `corner` (0 south, 1 east, 2 north, 3 west), the fast
 * axis leaves the origin counter-clockwise (sense 0; seen from outside the sphere, S -> E -> N -> W) or clockwise (sense
 * 1) around the face, the slow axis the other way.  Fig. 3C's "counterclockwise from the south" is FLAT(0, 0) (col = x,
 * row = y of the NESTED face coordinates), "clockwise from the east" is FLAT(1, 1) (reading R12; the paper
 * gives no formula).  Same argument conventions as cuhpx_reorder; RING <-> NESTED takes the tiled kernels of
 * cuhpx_reorder, every pair involving a flat layout one generic pass (reads or writes coalesced on the non-RING side). */
#define CUHPX_LAYOUT_RING 0
#define CUHPX_LAYOUT_NESTED 1
#define CUHPX_LAYOUT_FLAT(corner, sense) (2 + 2 * (corner) + (sense))
int cuhpx_reorder_layout(int nside, int batch, cuhpx_dtype_t dtype, int src_layout, int dst_layout, const void* d_in,
                         void* d_out, cuhpx_stream_t stream);
/* host helper: index in dst_layout of the pixel with index ip_src in src_layout (src_layout must not be RING); -1 on bad arguments */
long long cuhpx_layout_index(int nside, int src_layout, int dst_layout, long long ip_src);
/* host helper: RING index of NESTED pixel ipnest; -1 on bad arguments */
long long cuhpx_nest2ring_index(int nside, long long ipnest);

/* ---- spectral resampling ("upsampling and downsampling ... by truncating or extending
 * spherical harmonic coefficients before applying the iSHT").  d_alm_out(l, m) = d_alm_in(l, m) for l <= lmax_in and
 * m <= mmax_in, 0 elsewhere; both arrays [batch][nalm] complex, m-major packed for their own (lmax, mmax), DEVICE
 * pointers, 16-byte aligned, no aliasing.  Resampling a map from nside_a to nside_b is then
 * cuhpx_map2alm (nside_a) -> cuhpx_alm_resize -> cuhpx_alm2map (nside_b). */
int cuhpx_alm_resize(int lmax_in, int mmax_in, int lmax_out, int mmax_out, int batch, cuhpx_dtype_t dtype,
                     const void* d_alm_in, void* d_alm_out, cuhpx_stream_t stream);

/* ---- the same transforms on iso-latitude grids (the two-stage structure "generalizes to
 * ... Legendre-Gauss or Lobatto grids", used there for regridding through torch-harmonics).  A grid is nlat rings, north
 * to south, of nlon equally spaced pixels each, the first at phi = 0; map layout [batch][nlat * nlon], ring-major.
 *   CUHPX_GRID_GAUSS_LEGENDRE: cos(theta_k) = the nlat roots of P_nlat, per-pixel weight w_k^GL 2 pi / nlon: analysis is
 *       exact for band limit lmax <= nlat - 1, mmax <= (nlon - 1) / 2, so map2alm(alm2map(a)) = a to rounding
 *   CUHPX_GRID_EQUIANGULAR:    theta_k = pi (k + 1/2) / nlat with Fejer's first-rule weights (exact for zonal
 *       polynomials of degree <= nlat - 1, i.e. a round trip is exact for lmax <= (nlat - 1) / 2)
 *   CUHPX_GRID_HEALPIX:        nlat = nside, nlon ignored: identical to the calls above
 * nlon must be a power of two, 4 <= nlon <= 16384; 1 <= nlat <= 16384.  d_ring_weights: nlat doubles or NULL = the grid's
 * own quadrature weights.  Every other convention (alm layout, ownership, workspace header, asynchrony, error codes,
 * adjoint inner products) is that of the HEALPix calls; the kernels are the same, only the ring table differs. */
size_t cuhpx_grid_npix(int grid, int nlat, int nlon);
/* cos(theta) and the per-pixel quadrature weight of ring 1 .. nlat (host only; not for CUHPX_GRID_HEALPIX: cuhpx_ring_info) */
int cuhpx_grid_ring_info(int grid, int nlat, int nlon, int ring, double* cos_theta, double* weight);
size_t cuhpx_grid_workspace_bytes(int grid, int nlat, int nlon, int lmax, int mmax, int batch, cuhpx_dtype_t dtype);
int cuhpx_grid_workspace_init(int grid, int nlat, int nlon, int lmax, int mmax, int batch, cuhpx_dtype_t dtype,
                              void* d_workspace, size_t workspace_bytes, cuhpx_stream_t stream);
int cuhpx_grid_alm2map(int grid, int nlat, int nlon, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, const void* d_alm,
                       void* d_map, void* d_workspace, size_t workspace_bytes, cuhpx_stream_t stream);
int cuhpx_grid_map2alm(int grid, int nlat, int nlon, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, const void* d_map,
                       void* d_alm, const double* d_ring_weights, void* d_workspace, size_t workspace_bytes,
                       cuhpx_stream_t stream);
int cuhpx_grid_alm2map_adjoint(int grid, int nlat, int nlon, int lmax, int mmax, int batch, cuhpx_dtype_t dtype,
                               const void* d_gmap, void* d_galm, void* d_workspace, size_t workspace_bytes,
                               cuhpx_stream_t stream);
int cuhpx_grid_map2alm_adjoint(int grid, int nlat, int nlon, int lmax, int mmax, int batch, cuhpx_dtype_t dtype,
                               const void* d_galm, void* d_gmap, const double* d_ring_weights, void* d_workspace,
                               size_t workspace_bytes, cuhpx_stream_t stream);

/* ---- the two stages of each direction, individually, for per-stage
 * measurement and stage-level parity tests; same conventions and checks as the operators.  The ring spectra live
 * inside the workspace at byte offset cuhpx_spectra_offset(...):
 *   spectra[b][ring][m], m = 0..m_cut(ring) (entries above m_cut(ring) are neither written nor read: there
 *   lambda_lm(theta_ring) is below 2^-110 for every l <= lmax), row stride cuhpx_spectra_stride() complex values.
 * analysis:  F_m(ring) = w_ring sum_x p_x exp(-i m (phi0 + 2 pi x / N))   (Eq. 13, phase and alias rule of Eq. 26)
 * synthesis: p_x = Re G_0 + 2 sum_{m>=1} Re(G_m exp(+i m (phi0 + 2 pi x / N))), times w_ring if weights are given. */
size_t cuhpx_spectra_stride(int mmax);
/* byte offset of the spectra buffer inside a workspace for these parameters (0 on invalid arguments) */
size_t cuhpx_spectra_offset(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype);
/* m_cut of every ring (host array of 4 nside - 1 ints); host only */
int cuhpx_plan_mcut(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, int* h_mcut);
int cuhpx_analysis_fft_stage(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, const void* d_map,
                             const double* d_ring_weights, int use_weights, void* d_workspace, size_t workspace_bytes,
                             cuhpx_stream_t stream);
/* adjoint != 0 multiplies by c_m (S^T) */
int cuhpx_analysis_legendre_stage(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, void* d_alm, int adjoint,
                                  void* d_workspace, size_t workspace_bytes, cuhpx_stream_t stream);
/* adjoint != 0 divides the input by c_m (A^T) */
int cuhpx_synthesis_legendre_stage(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, const void* d_alm,
                                   int adjoint, void* d_workspace, size_t workspace_bytes, cuhpx_stream_t stream);
int cuhpx_synthesis_fft_stage(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, void* d_map,
                              const double* d_ring_weights, int use_weights, void* d_workspace, size_t workspace_bytes,
                              cuhpx_stream_t stream);

/* Host-side statistics of the plan for these parameters, for measurement (doubles, `count` of them are written, at most 8):
 *  [0] kernel launches of one FFT-stage call   [1] of one Legendre analysis call   [2] of one Legendre synthesis call
 *  [3] Legendre terms executed per channel = sum_m (lmax - m + 1) * (ring pairs processed at order m)
 *  [4] Legendre terms of the full triangle = nalm * 2 nside          [5] spectra entries per channel = sum_rings (m_cut + 1)
 *  [6] bytes of constant tables read by one FFT-stage call (chirp filters + twiddles)   [7] workspace bytes */
int cuhpx_plan_stats(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, double* h_stats, int count);

/* Measurement companion of cuhpx_plan_stats for an initialised workspace: h_skipped[0] / h_skipped[1] = Legendre steps
 * ((m, ring pair, degree) triples counted in [3] above) that the fp64 analysis / synthesis kernels do NOT walk because of
 * the late-start tables (0 when none are planned, see CUHPX_LATE_START).  Reads the tables back: SYNCHRONISES `stream`. */
int cuhpx_late_start_stats(int nside, int lmax, int mmax, int batch, cuhpx_dtype_t dtype, const void* d_workspace,
                           size_t workspace_bytes, cuhpx_stream_t stream, double* h_skipped);

/* MEASUREMENT HOOK, not part of the transform API: register-only FMA loop used by bench.py to measure the FP64 /
 * FP32 FMA peak of the device in the same run as the transforms (SURVEY 8(d) asks for exactly that).
 * Writes the elapsed milliseconds of `iters` dependent-chain FMAs per thread over the whole GPU to *ms and the
 * number of FMA instructions executed to *fma_count.  Synchronises the stream. */
int cuhpx_fma_peak_probe(cuhpx_dtype_t dtype, int iters, float* ms, double* fma_count, cuhpx_stream_t stream);

#ifdef __cplusplus
}
#endif
#endif /* CUHPX_H_ */

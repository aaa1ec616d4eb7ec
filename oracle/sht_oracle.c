/*
 * sht_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU oracle for the HEALPix RING spherical harmonic transform of
 * cuHPX (arXiv 2510.01785; /root/reference/PAPER.md, cited below as P:<line>).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call this file.
 * It shares no code, header, table or constant generator with the CUDA path under
 * paper_2510_01785_b200/csrc/, and neither includes the other.
 *
 * What it computes (the plain defining sums, no FFT, no north/south pairing, no fold, no skipping):
 *   synthesis  S  (alm2map)          Eq. 24
 *   analysis   A  (map2alm)          Eq. 26, P:277  (a = Y^dagger W p, Eq. 27)
 *   S^T (alm2map_adjoint), A^T (map2alm_adjoint)     P:286-292, transposes w.r.t. the real inner
 *   products <f,g> = sum_p f_p g_p and <a,b> = sum_{l, m>=0} (Re a Re b + Im a Im b)
 *   (reading R4: the inner product PyTorch autograd uses for the stored m>=0 tensor).
 *
 * Arithmetic: x87 80-bit `long double` throughout (recurrence, twiddles, accumulators); results are
 * rounded to double on output.  lambda_lm carries an explicit power-of-two exponent, because
 * sin^m(theta) underflows even long double at nside 4096 (SURVEY 7 "Underflow").
 *
 * Geometry (reading R1; formulas from Gorski et al., ref [1] P:416; counts P:94-96):
 *   rings i = 1 .. 4*nside-1 north->south, i' = min(i, 4 nside - i)
 *   polar cap  i' <  nside : N_i = 4 i', z = +-(1 - i'^2/(3 nside^2)), phi0 = pi/N_i
 *   belt nside<=i<=3nside   : N_i = 4 nside, z = 4/3 - 2 i/(3 nside), phi0 = pi/N_i if (i-nside) even else 0
 *   pixel x of ring i sits at phi = phi0 + 2 pi x / N_i, RING index = start_i + x
 *
 * lambda_lm (Eq. 15 P:195 with the explicit Condon-Shortley (-1)^m; Eq. 16 P:200 three-term recurrence;
 * cos(theta) enters as sgn*(1 - y) with y = 1 - |cos theta| formed exactly from the ring integers, because
 * cos(theta) rounded to any fixed precision loses theta near the poles -- DESIGN.md reading R3):
 *   lambda_00 = 1/sqrt(4 pi);  lambda_mm = -sqrt((2m+1)/(2m)) sin(theta) lambda_{m-1,m-1}
 *   lambda_{m+1,m} = sqrt(2m+3) cos(theta) lambda_mm
 *   lambda_lm = a cos(theta) lambda_{l-1,m} + b lambda_{l-2,m},
 *       a = sqrt((4l^2-1)/(l^2-m^2)),  b = -sqrt((2l+1)/(2l-3) * ((l-1)^2-m^2)/(l^2-m^2))
 *
 * alm layout: m-major packed, index(l,m) = m(2 lmax + 1 - m)/2 + l, complex interleaved (re,im),
 * m = 0..mmax, l = m..lmax (reading R5).
 *
 * Pins: tests/test_oracle_pins.py (closed forms, scipy sph_harm_y, mpmath, addition theorem,
 * Gauss-Legendre orthonormality, dense brute-force matrices, dot-product identities, geometry facts).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double ld;

#define ORACLE_OK 0
#define ORACLE_EINVAL 1
#define ORACLE_ENOMEM 2

static const ld PI_L = 3.14159265358979323846264338327950288419716939937510L;

/* ------------------------------------------------------------------ geometry (A1) */

typedef struct {
    int64_t n;      /* pixels in ring, N_i */
    int64_t start;  /* RING index of first pixel */
    ld z;           /* cos(theta_i) */
    ld y;           /* 1 - |cos(theta_i)|, formed without cancellation */
    ld sth;         /* sin(theta_i) */
    int shifted;    /* 1: phi0 = pi/N_i, 0: phi0 = 0 */
} ring_t;

static int is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }

static int ring_geometry(int nside, int i, ring_t* r) {
    if (!is_pow2(nside) || i < 1 || i > 4 * nside - 1) return ORACLE_EINVAL;
    const int64_t ns = nside;
    const int64_t npix = 12 * ns * ns;
    const int south = i > 2 * nside;
    const int64_t ip = south ? 4 * ns - i : i; /* northern mirror ring */
    ld z, one_minus_z;
    int64_t start;
    if (ip < ns) { /* polar cap */
        r->n = 4 * ip;
        one_minus_z = (ld)(ip * ip) / (ld)(3 * ns * ns);
        z = 1.0L - one_minus_z;
        r->y = one_minus_z;
        r->shifted = 1;
        start = 2 * ip * (ip - 1);
        r->sth = sqrtl(one_minus_z * (1.0L + z));
    } else { /* equatorial belt (northern half incl. equator) */
        r->n = 4 * ns;
        z = (ld)(4 * ns - 2 * ip) / (ld)(3 * ns);
        r->y = (ld)(2 * ip - ns) / (ld)(3 * ns);
        r->shifted = ((ip - ns) % 2 == 0) ? 1 : 0;
        start = 2 * ns * (ns - 1) + (ip - ns) * 4 * ns;
        r->sth = sqrtl((1.0L - z) * (1.0L + z));
    }
    if (south) {
        z = -z;
        start = npix - r->n - start;
    }
    r->z = z;
    r->start = start;
    return ORACLE_OK;
}

int oracle_ring_geometry(int nside, int ring, int64_t* n, int64_t* start, double* cos_theta,
                         double* sin_theta, double* phi0) {
    ring_t r;
    int rc = ring_geometry(nside, ring, &r);
    if (rc) return rc;
    *n = r.n;
    *start = r.start;
    *cos_theta = (double)r.z;
    *sin_theta = (double)r.sth;
    *phi0 = r.shifted ? (double)(PI_L / (ld)r.n) : 0.0;
    return ORACLE_OK;
}

int64_t oracle_alm_count(int lmax, int mmax) {
    return (int64_t)(mmax + 1) * (lmax + 1) - (int64_t)mmax * (mmax + 1) / 2;
}

static inline int64_t alm_index(int lmax, int l, int m) {
    return (int64_t)m * (2 * (int64_t)lmax + 1 - m) / 2 + l;
}

int64_t oracle_alm_index(int lmax, int l, int m) { return alm_index(lmax, l, m); }

/* ------------------------------------------------------------------ lambda_lm (A2) */

/* scaled value: true = v * 2^e */
typedef struct {
    ld v;
    long e;
} sld;

static inline void sld_norm(sld* s) {
    if (s->v != 0.0L) {
        int ex;
        s->v = frexpl(s->v, &ex);
        s->e += ex;
    }
}

/* lambda_00 = 1/sqrt(4 pi) */
static sld seed_00(void) {
    sld s = {1.0L / sqrtl(4.0L * PI_L), 0};
    sld_norm(&s);
    return s;
}

/* lambda_mm from lambda_{m-1,m-1}: times -sqrt((2m+1)/(2m)) sin(theta) */
static inline void seed_step(sld* s, int m, ld sth) {
    s->v *= -sqrtl((ld)(2 * m + 1) / (ld)(2 * m)) * sth;
    sld_norm(s);
}

/* Fill lam[l - m] = lambda_lm(theta) for l = m .. lmax (true values as long double; entries whose
 * magnitude is below the long double range come out as 0, which is far below anything a double
 * result can see).  seed = lambda_mm as a scaled value. */
static void lambda_column(int lmax, int m, ld y, int south, sld seed, ld* lam) {
    /* x * p is formed as +-(p - y p): see the header note on cos(theta) near the poles */
#define XMUL(p) (south ? -((p) - y * (p)) : ((p) - y * (p)))
    const long BIG = 8000; /* renormalise when the running pair leaves 2^+-8000 */
    ld p2 = seed.v; /* lambda_{l-2} mantissa */
    long e = seed.e; /* common exponent of the running pair */
    lam[0] = ldexpl(p2, (int)(e < -40000 ? -40000 : e));
    if (lmax == m) return;
    ld p1 = sqrtl((ld)(2 * m + 3)) * XMUL(p2); /* lambda_{m+1,m} */
    lam[1] = ldexpl(p1, (int)(e < -40000 ? -40000 : e));
    const ld m2 = (ld)m * (ld)m;
    for (int l = m + 2; l <= lmax; ++l) {
        const ld l2 = (ld)l * (ld)l;
        const ld a = sqrtl((4.0L * l2 - 1.0L) / (l2 - m2));
        const ld lm1 = (ld)(l - 1);
        const ld b = -sqrtl(((ld)(2 * l + 1) / (ld)(2 * l - 3)) * ((lm1 * lm1 - m2) / (l2 - m2)));
        const ld p0 = a * XMUL(p1) + b * p2;
        p2 = p1;
        p1 = p0;
        ld mag = fabsl(p1) > fabsl(p2) ? fabsl(p1) : fabsl(p2);
        if (mag > ldexpl(1.0L, BIG)) {
            p1 = ldexpl(p1, -BIG);
            p2 = ldexpl(p2, -BIG);
            e += BIG;
        } else if (mag != 0.0L && mag < ldexpl(1.0L, -BIG)) {
            p1 = ldexpl(p1, BIG);
            p2 = ldexpl(p2, BIG);
            e -= BIG;
        }
        lam[l - m] = ldexpl(p1, (int)(e < -40000 ? -40000 : e));
    }
#undef XMUL
}

/* Public: lambda_lm(theta) for l = 0..lmax at one colatitude (entries l < m are 0). */
int oracle_lambda(int lmax, int m, double theta, double* out) {
    if (lmax < 0 || m < 0 || m > lmax) return ORACLE_EINVAL;
    const ld sth = sinl((ld)theta);
    const int south = (ld)theta > PI_L / 2.0L;
    const ld half = south ? (PI_L - (ld)theta) / 2.0L : (ld)theta / 2.0L;
    const ld y = 2.0L * sinl(half) * sinl(half); /* 1 - |cos theta| */
    sld s = seed_00();
    for (int k = 1; k <= m; ++k) seed_step(&s, k, sth);
    ld* lam = (ld*)malloc(sizeof(ld) * (size_t)(lmax - m + 1));
    if (!lam) return ORACLE_ENOMEM;
    lambda_column(lmax, m, y, south, s, lam);
    for (int l = 0; l < m; ++l) out[l] = 0.0;
    for (int l = m; l <= lmax; ++l) out[l] = (double)lam[l - m];
    free(lam);
    return ORACLE_OK;
}

/* Public: lambda_lm at HEALPix ring `ring` of `nside` (uses the long double ring colatitude). */
int oracle_lambda_ring(int nside, int ring, int lmax, int m, double* out) {
    ring_t r;
    int rc = ring_geometry(nside, ring, &r);
    if (rc) return rc;
    if (lmax < 0 || m < 0 || m > lmax) return ORACLE_EINVAL;
    sld s = seed_00();
    for (int k = 1; k <= m; ++k) seed_step(&s, k, r.sth);
    ld* lam = (ld*)malloc(sizeof(ld) * (size_t)(lmax - m + 1));
    if (!lam) return ORACLE_ENOMEM;
    lambda_column(lmax, m, r.y, r.z < 0.0L, s, lam);
    for (int l = 0; l < m; ++l) out[l] = 0.0;
    for (int l = m; l <= lmax; ++l) out[l] = (double)lam[l - m];
    free(lam);
    return ORACLE_OK;
}

/* ------------------------------------------------------------------ ring DFT (A3) */

/* Table of exp(i pi j / n) for j = 0 .. 2n-1: the angle m (phi0 + 2 pi x / N) with phi0 = s pi / N
 * equals pi (m s + 2 m x) / N, so every twiddle is an exact integer index into this table. */
static int twiddle_table(int64_t n, ld** c, ld** s) {
    *c = (ld*)malloc(sizeof(ld) * (size_t)(2 * n));
    *s = (ld*)malloc(sizeof(ld) * (size_t)(2 * n));
    if (!*c || !*s) return ORACLE_ENOMEM;
    for (int64_t j = 0; j < 2 * n; ++j) {
        (*c)[j] = cosl(PI_L * (ld)j / (ld)n);
        (*s)[j] = sinl(PI_L * (ld)j / (ld)n);
    }
    return ORACLE_OK;
}

/* F_m = sum_x p_x exp(-i m (phi0 + 2 pi x / N)),  m = 0..mmax   (Eq. 13 P:177 / Eq. 26) */
static void ring_analysis_dft(const ring_t* r, const ld* tc, const ld* ts, const double* p, int mmax,
                              ld* Fre, ld* Fim) {
    const int64_t n = r->n, n2 = 2 * n;
    for (int m = 0; m <= mmax; ++m) {
        ld sr = 0.0L, si = 0.0L;
        int64_t idx = ((int64_t)m * r->shifted) % n2; /* x = 0 */
        const int64_t step = (2 * (int64_t)m) % n2;
        for (int64_t x = 0; x < n; ++x) {
            sr += (ld)p[x] * tc[idx];
            si -= (ld)p[x] * ts[idx];
            idx += step;
            if (idx >= n2) idx -= n2;
        }
        Fre[m] = sr;
        Fim[m] = si;
    }
}

/* p_x = Re G_0 + cm * sum_{m>=1} Re(G_m exp(+i m (phi0 + 2 pi x / N)))   (Eq. 24 P:267 with the
 * m<0 terms folded in by reality of the map, a_{l,-m} = (-1)^m conj(a_lm): cm = 2 for S). */
static void ring_synthesis_dft(const ring_t* r, const ld* tc, const ld* ts, const ld* Gre, const ld* Gim,
                               int mmax, ld cm, ld scale, double* p) {
    const int64_t n = r->n, n2 = 2 * n;
    for (int64_t x = 0; x < n; ++x) {
        ld acc = Gre[0];
        for (int m = 1; m <= mmax; ++m) {
            const int64_t idx = ((int64_t)m * r->shifted + 2 * (int64_t)m * x) % n2;
            acc += cm * (Gre[m] * tc[idx] - Gim[m] * ts[idx]);
        }
        p[x] = (double)(scale * acc);
    }
}

/* Public: the ring DFT alone (for the "FFT-free O(N^2) sum" pin and Bluestein-identity tests). */
int oracle_ring_dft(int nside, int ring, const double* p, int mmax, double* F /* (mmax+1) x (re,im) */) {
    ring_t r;
    int rc = ring_geometry(nside, ring, &r);
    if (rc) return rc;
    if (mmax < 0) return ORACLE_EINVAL;
    ld *tc, *ts;
    if (twiddle_table(r.n, &tc, &ts)) return ORACLE_ENOMEM;
    ld* Fre = (ld*)malloc(sizeof(ld) * (size_t)(mmax + 1));
    ld* Fim = (ld*)malloc(sizeof(ld) * (size_t)(mmax + 1));
    ring_analysis_dft(&r, tc, ts, p, mmax, Fre, Fim);
    for (int m = 0; m <= mmax; ++m) {
        F[2 * m] = (double)Fre[m];
        F[2 * m + 1] = (double)Fim[m];
    }
    free(Fre); free(Fim); free(tc); free(ts);
    return ORACLE_OK;
}

/* Public: the ring synthesis sum alone, p_x = Re G_0 + 2 sum_{m=1..mmax} Re(G_m exp(+i m (phi0 + 2 pi x / N))). */
int oracle_ring_synth(int nside, int ring, const double* G /* (mmax+1) x (re,im) */, int mmax, double* p) {
    ring_t r;
    int rc = ring_geometry(nside, ring, &r);
    if (rc) return rc;
    if (mmax < 0) return ORACLE_EINVAL;
    ld *tc, *ts;
    if (twiddle_table(r.n, &tc, &ts)) return ORACLE_ENOMEM;
    ld* Gre = (ld*)malloc(sizeof(ld) * (size_t)(mmax + 1));
    ld* Gim = (ld*)malloc(sizeof(ld) * (size_t)(mmax + 1));
    for (int m = 0; m <= mmax; ++m) {
        Gre[m] = (ld)G[2 * m];
        Gim[m] = (ld)G[2 * m + 1];
    }
    ring_synthesis_dft(&r, tc, ts, Gre, Gim, mmax, 2.0L, 1.0L, p);
    free(Gre); free(Gim); free(tc); free(ts);
    return ORACLE_OK;
}

/* ------------------------------------------------------------------ the four operators (A4) */

static int check_args(int nside, int lmax, int mmax) {
    if (!is_pow2(nside) || lmax < 0 || mmax < 0 || mmax > lmax) return ORACLE_EINVAL;
    return ORACLE_OK;
}

/* Generic synthesis-type sum over a list of rings:
 *   p_x(ring) = wscale_ring * [ sum_l Re(a_l0) lam_l0 + cm * sum_{m>=1} sum_l Re(a_lm lam_lm e^{i m phi_x}) ]
 * cm = 2, wscale = 1           -> S   (alm2map)
 * cm = 1, wscale = w_ring      -> A^T (map2alm_adjoint)
 * out: if `compact` the selected rings are written back to back, else at their RING offsets. */
static int synthesis_core(int nside, int lmax, int mmax, const double* alm, ld cm, const double* ring_w,
                          int use_w, int nsel, const int* sel_rings, int compact, double* out) {
    int rc = check_args(nside, lmax, mmax);
    if (rc) return rc;
    const int nrings = 4 * nside - 1;
    const int count = sel_rings ? nsel : nrings;
    const ld w_equal = 4.0L * PI_L / (12.0L * (ld)nside * (ld)nside);
    /* compact offsets */
    int64_t* coff = (int64_t*)malloc(sizeof(int64_t) * (size_t)(count + 1));
    if (!coff) return ORACLE_ENOMEM;
    coff[0] = 0;
    for (int k = 0; k < count; ++k) {
        ring_t r;
        rc = ring_geometry(nside, sel_rings ? sel_rings[k] : k + 1, &r);
        if (rc) { free(coff); return rc; }
        coff[k + 1] = coff[k] + r.n;
    }
    int fail = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < count; ++k) {
        const int ring = sel_rings ? sel_rings[k] : k + 1;
        ring_t r;
        ring_geometry(nside, ring, &r);
        ld *tc = NULL, *ts = NULL;
        ld* lam = (ld*)malloc(sizeof(ld) * (size_t)(lmax + 1));
        ld* Gre = (ld*)malloc(sizeof(ld) * (size_t)(mmax + 1));
        ld* Gim = (ld*)malloc(sizeof(ld) * (size_t)(mmax + 1));
        if (!lam || !Gre || !Gim || twiddle_table(r.n, &tc, &ts)) {
#pragma omp atomic write
            fail = 1;
        } else {
            sld seed = seed_00();
            for (int m = 0; m <= mmax; ++m) {
                if (m > 0) seed_step(&seed, m, r.sth);
                lambda_column(lmax, m, r.y, r.z < 0.0L, seed, lam);
                const double* a = alm + 2 * alm_index(lmax, m, m);
                ld gr = 0.0L, gi = 0.0L;
                for (int l = m; l <= lmax; ++l) {
                    gr += (ld)a[2 * (l - m)] * lam[l - m];
                    if (m > 0) gi += (ld)a[2 * (l - m) + 1] * lam[l - m]; /* Im a_l0 ignored */
                }
                Gre[m] = gr;
                Gim[m] = gi;
            }
            ld scale = 1.0L;
            if (use_w) scale = ring_w ? (ld)ring_w[ring - 1] : w_equal;
            double* dst = compact ? out + coff[k] : out + r.start;
            ring_synthesis_dft(&r, tc, ts, Gre, Gim, mmax, cm, scale, dst);
        }
        free(lam); free(Gre); free(Gim); free(tc); free(ts);
    }
    free(coff);
    return fail ? ORACLE_ENOMEM : ORACLE_OK;
}

/* Generic analysis-type sum:
 *   a_lm = cfac_m * sum_rings wscale_ring * lam_lm(theta_ring) * sum_x p_x e^{-i m phi_x}
 * cfac = 1, wscale = w_ring  -> A   (map2alm)
 * cfac = c_m (1 for m = 0, 2 otherwise), wscale = 1 -> S^T (alm2map_adjoint)
 * If sel_l/sel_m are given only those nsel coefficients are computed (out is nsel x (re,im)),
 * otherwise the full packed alm array. */
static int analysis_core(int nside, int lmax, int mmax, const double* map, const double* ring_w, int use_w,
                         int double_m, int nsel, const int* sel_l, const int* sel_m, double* out) {
    int rc = check_args(nside, lmax, mmax);
    if (rc) return rc;
    const int nrings = 4 * nside - 1;
    const ld w_equal = 4.0L * PI_L / (12.0L * (ld)nside * (ld)nside);
    const int64_t nalm = oracle_alm_count(lmax, mmax);
    const int64_t nout = sel_l ? nsel : nalm;
    /* per-m flags and (for subsets) the largest l wanted for that m */
    int* want_lmax = (int*)malloc(sizeof(int) * (size_t)(mmax + 1));
    if (!want_lmax) return ORACLE_ENOMEM;
    for (int m = 0; m <= mmax; ++m) want_lmax[m] = sel_l ? -1 : lmax;
    if (sel_l) {
        for (int k = 0; k < nsel; ++k) {
            if (sel_m[k] < 0 || sel_m[k] > mmax || sel_l[k] < sel_m[k] || sel_l[k] > lmax) {
                free(want_lmax);
                return ORACLE_EINVAL;
            }
            if (sel_l[k] > want_lmax[sel_m[k]]) want_lmax[sel_m[k]] = sel_l[k];
        }
    }
    int nthreads = 1;
#ifdef _OPENMP
    nthreads = omp_get_max_threads();
#endif
    ld* acc = (ld*)calloc((size_t)nthreads * (size_t)nout * 2, sizeof(ld));
    if (!acc) { free(want_lmax); return ORACLE_ENOMEM; }
    int fail = 0;
#pragma omp parallel
    {
        int tid = 0;
#ifdef _OPENMP
        tid = omp_get_thread_num();
#endif
        ld* my = acc + (size_t)tid * (size_t)nout * 2;
        ld* lam = (ld*)malloc(sizeof(ld) * (size_t)(lmax + 1));
        ld* Fre = (ld*)malloc(sizeof(ld) * (size_t)(mmax + 1));
        ld* Fim = (ld*)malloc(sizeof(ld) * (size_t)(mmax + 1));
        if (!lam || !Fre || !Fim) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp for schedule(dynamic, 1)
        for (int ring = 1; ring <= nrings; ++ring) {
            if (fail) continue;
            ring_t r;
            ring_geometry(nside, ring, &r);
            ld *tc = NULL, *ts = NULL;
            if (twiddle_table(r.n, &tc, &ts)) {
#pragma omp atomic write
                fail = 1;
                free(tc); free(ts);
                continue;
            }
            const double* p = map + r.start;
            ld w = 1.0L;
            if (use_w) w = ring_w ? (ld)ring_w[ring - 1] : w_equal;
            if (!sel_l) {
                ring_analysis_dft(&r, tc, ts, p, mmax, Fre, Fim);
            } else { /* only the wanted m */
                const int64_t n = r.n, n2 = 2 * n;
                for (int m = 0; m <= mmax; ++m) {
                    if (want_lmax[m] < 0) continue;
                    ld sr = 0.0L, si = 0.0L;
                    int64_t idx = ((int64_t)m * r.shifted) % n2;
                    const int64_t step = (2 * (int64_t)m) % n2;
                    for (int64_t x = 0; x < n; ++x) {
                        sr += (ld)p[x] * tc[idx];
                        si -= (ld)p[x] * ts[idx];
                        idx += step;
                        if (idx >= n2) idx -= n2;
                    }
                    Fre[m] = sr;
                    Fim[m] = si;
                }
            }
            sld seed = seed_00();
            for (int m = 0; m <= mmax; ++m) {
                if (m > 0) seed_step(&seed, m, r.sth);
                if (want_lmax[m] < 0) continue;
                lambda_column(want_lmax[m], m, r.y, r.z < 0.0L, seed, lam);
                const ld cf = (double_m && m > 0) ? 2.0L : 1.0L;
                const ld fr = cf * w * Fre[m], fi = cf * w * Fim[m];
                if (!sel_l) {
                    ld* a = my + 2 * alm_index(lmax, m, m);
                    for (int l = m; l <= lmax; ++l) {
                        a[2 * (l - m)] += lam[l - m] * fr;
                        a[2 * (l - m) + 1] += lam[l - m] * fi;
                    }
                } else {
                    for (int k = 0; k < nsel; ++k)
                        if (sel_m[k] == m) {
                            my[2 * k] += lam[sel_l[k] - m] * fr;
                            my[2 * k + 1] += lam[sel_l[k] - m] * fi;
                        }
                }
            }
            free(tc); free(ts);
        }
        free(lam); free(Fre); free(Fim);
    }
    if (!fail) {
        for (int64_t k = 0; k < nout; ++k) {
            ld sr = 0.0L, si = 0.0L;
            for (int t = 0; t < nthreads; ++t) {
                sr += acc[(size_t)t * (size_t)nout * 2 + 2 * k];
                si += acc[(size_t)t * (size_t)nout * 2 + 2 * k + 1];
            }
            out[2 * k] = (double)sr;
            out[2 * k + 1] = (double)si;
        }
        /* Im a_l0 is exactly zero (sin(0) = 0 in the defining sum) */
        if (!sel_l) {
            for (int l = 0; l <= lmax; ++l) out[2 * alm_index(lmax, l, 0) + 1] = 0.0;
        } else {
            for (int k = 0; k < nsel; ++k)
                if (sel_m[k] == 0) out[2 * k + 1] = 0.0;
        }
    }
    free(acc);
    free(want_lmax);
    return fail ? ORACLE_ENOMEM : ORACLE_OK;
}

/* S: alm2map.  Eq. 24 P:267. */
int oracle_alm2map(int nside, int lmax, int mmax, const double* alm, double* map) {
    return synthesis_core(nside, lmax, mmax, alm, 2.0L, NULL, 0, 0, NULL, 0, map);
}

/* A: map2alm.  Eq. 26; ring_w = NULL means equal weights 4 pi / Npix (Eq. 1). */
int oracle_map2alm(int nside, int lmax, int mmax, const double* map, const double* ring_w, double* alm) {
    return analysis_core(nside, lmax, mmax, map, ring_w, 1, 0, 0, NULL, NULL, alm);
}

/* S^T: alm2map_adjoint ("adjoint iSHT = Y^dagger"), (S^T g)_lm = c_m sum_p g_p lam_lm e^{-i m phi_p}. */
int oracle_alm2map_adjoint(int nside, int lmax, int mmax, const double* gmap, double* galm) {
    return analysis_core(nside, lmax, mmax, gmap, NULL, 0, 1, 0, NULL, NULL, galm);
}

/* A^T: map2alm_adjoint ("adjoint SHT = W Y"),
 * (A^T b)_p = w_p [ sum_l Re(b_l0) lam_l0 + sum_{m>=1} sum_l Re(b_lm lam_lm e^{i m phi_p}) ]. */
int oracle_map2alm_adjoint(int nside, int lmax, int mmax, const double* galm, const double* ring_w,
                           double* gmap) {
    return synthesis_core(nside, lmax, mmax, galm, 1.0L, ring_w, 1, 0, NULL, 0, gmap);
}

/* Subset mode: selected coefficients of A / S^T, selected rings of S / A^T. */
int oracle_map2alm_subset(int nside, int lmax, int mmax, const double* map, const double* ring_w, int nsel,
                          const int* sel_l, const int* sel_m, double* out) {
    return analysis_core(nside, lmax, mmax, map, ring_w, 1, 0, nsel, sel_l, sel_m, out);
}

int oracle_alm2map_adjoint_subset(int nside, int lmax, int mmax, const double* gmap, int nsel, const int* sel_l,
                                  const int* sel_m, double* out) {
    return analysis_core(nside, lmax, mmax, gmap, NULL, 0, 1, nsel, sel_l, sel_m, out);
}

/* out holds the selected rings back to back, in the order given. */
int oracle_alm2map_rings(int nside, int lmax, int mmax, const double* alm, int nsel, const int* rings,
                         double* out) {
    return synthesis_core(nside, lmax, mmax, alm, 2.0L, NULL, 0, nsel, rings, 1, out);
}

int oracle_map2alm_adjoint_rings(int nside, int lmax, int mmax, const double* galm, const double* ring_w,
                                 int nsel, const int* rings, double* out) {
    return synthesis_core(nside, lmax, mmax, galm, 1.0L, ring_w, 1, nsel, rings, 1, out);
}

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
